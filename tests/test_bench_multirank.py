"""bench.py's N > 1 path on CPU: world_size 2 over gloo.  The path shards by independent problems (DESIGN.md
"Multi-GPU"): rank r owns the network of generator seed r, there is no data-path collective, times are reduced with
MAX and counts with SUM.  The GPU kernels are not involved here."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    net, params = bench.rank_problem("small", rank, 512)
    times = [10.0 + rank, 100.0 - rank]               # rank-dependent so that MAX and SUM are distinguishable
    counts = [float(net.S.shape[1]), float(rank + 1), 7.0]
    red = bench.reduce_over_ranks(times, counts, dist, torch.device("cpu"))
    cap = bench.agreed_cap(1 << (24 - rank), dist, torch.device("cpu"))   # rank 1 "fell back" one size
    dist.barrier()
    out[rank] = (red, int(np.abs(net.S).sum()), params["frontier_cap"], cap)
    dist.destroy_process_group()


def test_replica_reduction_world_size_2():
    world, port = 2, 29500 + os.getpid() % 2000
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
    r0, r1 = out[0], out[1]
    assert r0[0] == r1[0]                              # every rank sees the same whole-job figures
    t_a, t_b, c_a, c_b, c_c = r0[0]
    assert (t_a, t_b) == (11.0, 100.0)                 # MAX over ranks
    assert (c_a, c_b, c_c) == (64.0, 3.0, 14.0)        # SUM over ranks (32 reactions per small network)
    assert r0[1] != r1[1]                              # different generator seeds: independent problems
    assert r0[2] == r1[2] == 512
    assert r0[3] == r1[3] == 1 << 23                   # every rank times the smallest beam any rank fell back to


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks([1.5, 2.5], [3.0], None, torch.device("cpu")) == [1.5, 2.5, 3.0]
    assert bench.agreed_cap(1 << 22, None, torch.device("cpu")) == 1 << 22
