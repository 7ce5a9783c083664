"""Host-side logic of the N > 1 bench path (tier rule 5: the path does not shard, `bench.py --gpus N` runs N independent
spills): every rank draws its own seeded workload, the whole-job time is the max over ranks and the work the sum.
Runs on CPU with the gloo backend, world_size 2."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = bench.make_workload(0, rank)
    ms, n_all = bench.reduce_over_ranks(10.0 + 5.0 * rank, wl.n_segments, world, torch.device("cpu"))
    out[rank] = (ms, n_all, wl.seed, wl.n_segments, float(wl.segments["xs"][0]))
    dist.barrier()
    dist.destroy_process_group()


def test_weak_scaling_reduction_world_size_2():
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    ms0, n0, seed0, nseg0, x0 = res[0]
    ms1, n1, seed1, nseg1, x1 = res[1]
    assert ms0 == ms1 == 15.0                          # max over ranks
    assert n0 == n1 == nseg0 + nseg1                   # whole-job work = sum over ranks
    assert seed0 != seed1 and x0 != x1                 # every rank simulates its own spill


def test_rank_workloads_are_seeded_and_reproducible():
    import bench
    a, b = bench.make_workload(1, 3), bench.make_workload(1, 3)
    c = bench.make_workload(1, 0)
    for k in a.segments:
        assert np.array_equal(a.segments[k], b.segments[k])
    assert a.seed != c.seed and not np.array_equal(a.segments["xs"][:50], c.segments["xs"][:50])
