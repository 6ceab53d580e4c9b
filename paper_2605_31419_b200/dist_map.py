"""Sharding of a mapping step over ranks (the mapping window of several
keyframes).  The map is replicated; the keyframes of the window are dealt to the ranks; every rank accumulates the
per-vertex gradients of its own views with ts_render_map_l1 into ONE flat buffer, and one all-reduce (sum) of that
buffer per step merges them (NCCL over NVLink on GPUs, gloo in the CPU tests).  Plumbing only: no method arithmetic."""
from __future__ import annotations


def shard_views(n_views: int, rank: int, world: int) -> list[int]:
    """Views of rank `rank`: round-robin, so that neighbouring keyframes (similar cost) land on different ranks."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank / world size")
    return list(range(rank, n_views, world))


class GradBucket:
    """grad_pos [V,3], grad_color [V,3], grad_opacity [V] as views of one flat float32 buffer of 7 V elements: the
    all-reduce of a step is a single collective call."""

    def __init__(self, V: int, device):
        import torch
        self.V = int(V)
        self.flat = torch.zeros(7 * self.V, dtype=torch.float32, device=device)
        self.grad_pos = self.flat[: 3 * self.V].view(self.V, 3)
        self.grad_color = self.flat[3 * self.V: 6 * self.V].view(self.V, 3)
        self.grad_opacity = self.flat[6 * self.V:]

    def zero_(self):
        self.flat.zero_()

    def all_reduce(self, dist, async_op: bool = False):
        """Sum over ranks (no-op without a process group).  Returns the work handle when async_op is set."""
        if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
            return None
        return dist.all_reduce(self.flat, op=dist.ReduceOp.SUM, async_op=async_op)
