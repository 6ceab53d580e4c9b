"""World-size-2 gloo test (CPU) of bench.py's N > 1 host logic: the path is "replicas only", so
what has to be right is the rank -> frame assignment and the max-over-ranks reduction of the device-timed step."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2605_31419_b200 import scenes
    seed = bench.rank_seed(0, rank)
    sc = scenes.config0(n_faces=50, seed=seed)
    local_ms = 1.0 + rank                       # rank 1 is the slow one
    mx = bench.max_over_ranks(dist, local_ms, "cpu")
    checksum = float(np.abs(sc.pos).sum())
    gathered = [None] * world
    dist.all_gather_object(gathered, (seed, checksum, mx))
    if rank == 0:
        torch.save(gathered, out)
    dist.destroy_process_group()


def test_two_rank_replicas_gloo(tmp_path):
    out = str(tmp_path / "res.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    res = torch.load(out, weights_only=False)
    (s0, c0, m0), (s1, c1, m1) = res
    assert (s0, s1) == (0, 100)                 # every rank tracks its own frame
    assert c0 != c1
    assert m0 == m1 == 2.0                      # the step time reported is the max over ranks


def _map_worker(rank, world, port, out):
    """One rank of a sharded mapping step on CPU tensors: the oracle's gradients of this rank's views accumulated into
    the flat bucket, then the step's one all-reduce (gloo here, NCCL on GPUs): same plumbing as bench.py --config 3."""
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import tso
    from paper_2605_31419_b200 import dist_map, scenes
    sc = scenes.config3(n_faces=3000, n_views=5)
    sc.cam = scenes.Camera(160, 96, 80.0, 80.0, 79.5, 47.5)
    bucket = dist_map.GradBucket(sc.pos.shape[0], "cpu")
    mine = dist_map.shard_views(len(sc.T_gt), rank, world)
    for v in mine:
        tgt = tso.Oracle(sc.pos_target, sc.color_target, sc.opacity, None, sc.T_gt[v], sc.cam, sc.params, "f32").forward("tiled")
        o = tso.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_start[v], sc.cam, sc.params, "f32")
        f = o.forward("tiled")
        L, gC, gD = o.l1_loss(f.color, f.depth, tgt.color, tgt.depth, sc.params.lambda_dep)
        g = o.backward(gC, gD, None, want=("pos", "color", "opacity"))
        bucket.grad_pos += torch.from_numpy(g.grad_pos.astype(np.float32))
        bucket.grad_color += torch.from_numpy(g.grad_color.astype(np.float32))
        bucket.grad_opacity += torch.from_numpy(g.grad_opacity.astype(np.float32))
    local = bucket.flat.clone()
    bucket.all_reduce(dist)
    gathered = [None] * world
    dist.all_gather_object(gathered, (mine, local.numpy(), bucket.flat.numpy().copy()))
    if rank == 0:
        torch.save(gathered, out)
    dist.destroy_process_group()


def test_two_rank_sharded_mapping_step_gloo(tmp_path, oracle_mod):
    """views dealt to the ranks, replicated map, ONE all-reduce of the gradient buffer: the
    sharded sum equals the single-rank sum over all views (to float32 addition order)."""
    from paper_2605_31419_b200 import dist_map, scenes
    out = str(tmp_path / "map.pt")
    mp.spawn(_map_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    (v0, l0, r0), (v1, l1, r1) = torch.load(out, weights_only=False)
    assert sorted(v0 + v1) == [0, 1, 2, 3, 4] and not set(v0) & set(v1)      # every view on exactly one rank
    assert np.array_equal(r0, r1)                                              # both ranks hold the same sum afterwards
    assert np.abs(l0).max() > 0 and np.abs(l1).max() > 0
    # single rank, all views
    sc = scenes.config3(n_faces=3000, n_views=5)
    sc.cam = scenes.Camera(160, 96, 80.0, 80.0, 79.5, 47.5)
    ref = dist_map.GradBucket(sc.pos.shape[0], "cpu")
    for v in dist_map.shard_views(5, 0, 1):
        tgt = oracle_mod.Oracle(sc.pos_target, sc.color_target, sc.opacity, None, sc.T_gt[v], sc.cam, sc.params, "f32").forward("tiled")
        o = oracle_mod.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_start[v], sc.cam, sc.params, "f32")
        f = o.forward("tiled")
        L, gC, gD = o.l1_loss(f.color, f.depth, tgt.color, tgt.depth, sc.params.lambda_dep)
        g = o.backward(gC, gD, None, want=("pos", "color", "opacity"))
        ref.grad_pos += torch.from_numpy(g.grad_pos.astype(np.float32))
        ref.grad_color += torch.from_numpy(g.grad_color.astype(np.float32))
        ref.grad_opacity += torch.from_numpy(g.grad_opacity.astype(np.float32))
    want = ref.flat.numpy()
    assert np.abs(want).max() > 0
    assert np.abs(r0 - want).max() <= 1e-5 * np.abs(want).max()
    assert ref.all_reduce(None) is None                                        # no process group: a no-op


def test_shard_views_partitions():
    from paper_2605_31419_b200 import dist_map
    for n in (1, 5, 8):
        for w in (1, 2, 3, 8):
            if w > n:
                continue
            parts = [dist_map.shard_views(n, r, w) for r in range(w)]
            assert sorted(sum(parts, [])) == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
