"""-m "not gpu": the N > 1 plumbing of bench.py (max-over-ranks time, whole-job aggregate) on
world_size = 2 with the gloo backend.  The path shards by independent boxes: no data-path collective."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch
    import bench
    w, r, _ = bench.dist_setup(world, "gloo")
    assert (w, r) == (world, rank)
    dev = torch.device("cpu")
    ms = bench.all_max(10.0 + 5.0 * rank, dev)              # rank 1 is slower
    ns = bench.all_gather_int(1000 * (rank + 1), dev)
    bench.barrier()
    out[rank] = (ms, ns, bench.aggregate(ns, ms))
    import torch.distributed as dist
    dist.destroy_process_group()


def test_world2_gloo_aggregate():
    import torch.multiprocessing as mp
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in (0, 1):
        ms, ns, val = res[rank]
        assert ms == 15.0                                   # max over ranks
        assert ns == [1000, 2000]
        assert val == pytest.approx(3000 / 15e-3)           # units of all ranks / max time


def test_rank_workloads_are_independent_boxes():
    sys.path.insert(0, ROOT)
    import numpy as np
    import bench
    from paper_2606_17145_b200 import workloads as W
    a = W.uniform_box(8, 1.0, W.SEED0 + 1000)
    b = bench.make_workload("uniform32", 1)
    assert b.n == 32 ** 3 and not np.array_equal(a.pos[:8], b.pos[:8])
