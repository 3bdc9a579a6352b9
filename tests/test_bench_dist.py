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


# ---- strong scaling: Morton-range sharding of the active targets (paper_2606_17145_b200/sharding.py) -----------
def test_partition_by_cost_tiles_and_balances():
    sys.path.insert(0, ROOT)
    import numpy as np
    from paper_2606_17145_b200 import sharding as S
    rng = np.random.default_rng(0)
    for n, ranks in ((0, 4), (17, 4), (1000, 1), (100003, 8), (4096, 3)):
        cost = rng.integers(1, 1000, n)
        b = S.partition_by_cost(cost, ranks)
        assert b[0] == 0 and b[-1] == n and np.all(np.diff(b) >= 0)
        assert all(int(x) % S.ALIGN == 0 for x in b[1:-1])
        if n >= 50000:
            share = np.array([cost[b[r]:b[r + 1]].sum() for r in range(ranks)], dtype=np.float64)
            assert share.max() / share.mean() < 1.02
    # all-zero costs fall back to equal counts
    b = S.partition_by_cost(np.zeros(6400), 4)
    assert list(b) == [0, 1600, 3200, 4800, 6400]


def _strong_worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import numpy as np
    import torch
    import torch.distributed as dist
    import bench
    from paper_2606_17145_b200 import sharding as S
    bench.dist_setup(world, "gloo")
    # the same seeded problem on every rank: an active subset in arbitrary order (with one duplicate), slots, costs
    rng = np.random.default_rng(123)
    n = 20000
    inv_perm = rng.permutation(n).astype(np.uint32)                  # slot of every particle
    active = rng.choice(n, 5003, replace=False).astype(np.uint32)
    active[77] = active[5]
    cost = rng.integers(50, 2000, active.shape[0])
    order = S.sorted_active_order(inv_perm[active])
    bounds = S.partition_by_cost(cost[order], world)
    pos, idx = S.rank_sublist(active, n, order, bounds, rank)
    # stand-in for the walk: any function of the target alone (each target has one owner, no reduction)
    res = (idx.astype(np.float64) * 1.5 + 0.25)
    gathered = [None] * world
    dist.all_gather_object(gathered, (pos, res))
    full = np.full(active.shape[0], np.nan)
    seen = np.zeros(active.shape[0], np.int64)
    for p, r in gathered:
        full[p] = r
        seen[p] += 1
    out[rank] = (bool(np.all(seen == 1)), bool(np.array_equal(full, active.astype(np.float64) * 1.5 + 0.25)),
                 [int(x) for x in bounds])
    dist.destroy_process_group()


def test_world2_gloo_strong_sharding_tiles_the_active_set_once():
    import torch.multiprocessing as mp
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_strong_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    assert res[0][2] == res[1][2]                              # same boundaries on every rank
    for rank in (0, 1):
        once, equal, bounds = res[rank]
        assert once and equal
        assert bounds[0] == 0 and bounds[-1] == 5003 and bounds[1] % 32 == 0
