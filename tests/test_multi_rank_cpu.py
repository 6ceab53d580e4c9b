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
