"""-m "not gpu": the host layer of row f4 (paper_2606_17145_b200/let.py) on world_size = 2 with the gloo backend: the
splitter rule, the exchanges (all-reduce of the cell histogram, all-to-all of particles / targets / results with ragged
counts, all-gather of ragged box lists) and the order of the sums, with the device calls replaced by the oracle-backed
stand-in tests/let_stub.py.  The same pipeline run in ONE process with LocalExchange must give the same numbers, and
both must equal oracle.let.let_walk."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _problem():
    import oracle
    from paper_2606_17145_b200 import workloads as W
    w = W.nfw_box(16, 8, 100.0, W.SEED0 + 41, name="let_dist")
    prm = oracle.make_params(w.L, 2.5, alpha=w.alpha, theta=w.theta, leaf_max=8)
    rng = np.random.default_rng(3)
    a_old = (rng.random(w.n) * 0.02 + 1e-4).astype(np.float32)
    active = rng.random(w.n) < 0.6
    return w, prm, a_old, active


def _domains(w, a_old, active, ranks, world):
    import torch
    from paper_2606_17145_b200 import let
    out = {}
    for r in ranks:                                          # initial distribution: round robin, nothing to do with space
        sel = np.arange(r, w.n, world)
        out[r] = let.Domain(torch.from_numpy(w.pos[sel]), torch.from_numpy(w.mass[sel]), torch.from_numpy(w.eps[sel]),
                            torch.from_numpy(sel.astype(np.int64)), torch.from_numpy(active[sel]), torch.from_numpy(a_old[sel]))
    return out


def _run(ex, ranks, world):
    import let_stub
    from paper_2606_17145_b200 import let
    w, prm, a_old, active = _problem()
    doms, S = let.decompose(let_stub, _domains(w, a_old, active, ranks, world), ex, w.L)
    res, info = let.let_forces(let_stub, doms, ex, w.L, prm)
    return {r: (doms[r].gid[doms[r].active.long()].numpy(), res[r][0].numpy(), res[r][1].numpy(), doms[r].gid.numpy())
            for r in ranks}, S, info


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch.distributed as dist
    from paper_2606_17145_b200 import let
    dist.init_process_group("gloo", rank=rank, world_size=world)
    res, S, info = _run(let.DistExchange(), [rank], world)
    out[rank] = (res[rank], S, info["n_exported"])
    dist.destroy_process_group()


def test_splitters_hand_built():
    from paper_2606_17145_b200 import let
    h = np.zeros(let.N_CELLS, np.int64)
    h[[3, 10, 11, 500, 32767]] = [4, 1, 5, 6, 4]            # 20 particles; boundaries want 5, 10, 15 before them
    assert let.splitters(h, 4).tolist() == [0, 11, 12, 501, 32768]
    assert let.splitters(h, 1).tolist() == [0, 32768]
    assert let.splitters(np.zeros(let.N_CELLS, np.int64), 3).tolist() == [0, 0, 0, 32768]


def test_splitters_equal_the_oracle_rule_on_random_histograms():
    """paper_2606_17145_b200/let.py and oracle/let.py state R49 independently (searchsorted vs an explicit scan)."""
    from oracle import let as olet
    from paper_2606_17145_b200 import let
    rng = np.random.default_rng(77)
    for trial in range(40):
        h = np.zeros(let.N_CELLS, np.int64)
        k = int(rng.integers(1, 4000))
        cells = rng.choice(let.N_CELLS, size=k, replace=False)
        h[cells] = rng.integers(1, 10 ** int(rng.integers(1, 6)), size=k)
        for R in (1, 2, 3, 5, 8, 16, 64):
            S = let.splitters(h, R)
            assert np.array_equal(S, olet.splitters(h, R)), (trial, R)
            assert S[0] == 0 and S[-1] == let.N_CELLS and np.all(np.diff(S) >= 0)
            # balance: no domain exceeds its share by more than the largest cell
            per = np.add.reduceat(np.r_[h, 0], np.minimum(S[:-1], let.N_CELLS))[:R] * (np.diff(S) > 0)
            assert per.sum() == h.sum()
            assert per.max() <= -(-h.sum() // R) + h.max()


def test_world2_gloo_pipeline_equals_local_emulation_and_oracle():
    import torch.multiprocessing as mp
    import oracle
    from oracle import let as olet
    from paper_2606_17145_b200 import let
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        dist_res = dict(out)
    loc, S, info = _run(let.LocalExchange(2), [0, 1], 2)
    w, prm, a_old, active = _problem()
    act = np.flatnonzero(active).astype(np.uint32)
    a_ref, p_ref, oinfo = olet.let_walk(w.pos, w.mass, w.eps, prm, 2, active_idx=act, a_old=a_old[act])
    assert np.array_equal(S, oinfo["splitters"])
    pos_of = {int(g): k for k, g in enumerate(act)}
    seen = 0
    for r in (0, 1):
        (gid_a, acc, pot, gid_all), S_d, nexp = dist_res[r]
        assert np.array_equal(S_d, S)
        assert np.array_equal(np.sort(gid_all), np.flatnonzero(oinfo["owner"] == r))       # the right particles arrived
        assert np.array_equal(gid_a, loc[r][0]) and np.array_equal(acc, loc[r][1]) and np.array_equal(pot, loc[r][2])
        assert nexp[(r, 1 - r)] == oinfo["n_exported"][r, 1 - r] == info["n_exported"][(r, 1 - r)]
        k = np.array([pos_of[int(g)] for g in gid_a])
        assert np.abs(acc - a_ref[k]).max() <= 1e-5 * np.abs(a_ref).max()
        assert np.abs(pot - p_ref[k]).max() <= 1e-5 * np.abs(p_ref).max()
        seen += len(k)
    assert seen == len(act)
    assert 0 < oinfo["n_exported"].sum() < len(act)                                       # some, not all, are exported


def test_empty_domains_and_active_subset_local_emulation():
    """More domains than occupied level-5 cells: some domains own nothing (no tree, nothing exported to them); a sparse
    active subset; geometric criterion.  One process, oracle-backed stand-in, against oracle.let."""
    import torch
    import let_stub
    import oracle
    from oracle import let as olet
    from paper_2606_17145_b200 import let
    rng = np.random.default_rng(12)
    L = 10.0
    # three tight clumps: three occupied level-5 cells (side L / 32), 7 domains
    centres = np.array([[1.1, 1.1, 1.1], [1.3, 1.1, 1.1], [7.7, 3.3, 9.1]])
    pos = np.vstack([c + rng.random((40, 3)) * 0.05 for c in centres]).astype(np.float32)
    n = pos.shape[0]
    mass = (rng.random(n) + 0.5).astype(np.float32)
    eps = np.full(n, 1e-3, np.float32)
    prm = oracle.make_params(L, 0.2, alpha=0.005, theta=0.5, leaf_max=4)
    R = 7
    act = np.sort(rng.choice(n, 50, replace=False)).astype(np.uint32)
    mask = np.zeros(n, bool); mask[act] = True
    ex = let.LocalExchange(R)
    parts = {}
    for r in range(R):
        sel = np.arange(r, n, R)
        parts[r] = let.Domain(torch.from_numpy(pos[sel]), torch.from_numpy(mass[sel]), torch.from_numpy(eps[sel]),
                              torch.from_numpy(sel.astype(np.int64)), torch.from_numpy(mask[sel]), None)
    doms, S = let.decompose(let_stub, parts, ex, L)
    sizes = [int(doms[r].pos.shape[0]) for r in range(R)]
    assert sum(sizes) == n and sizes.count(0) >= 3                       # empty domains exist
    res, info = let.let_forces(let_stub, doms, ex, L, prm, geometric=True)
    a_ref, p_ref, oinfo = olet.let_walk(pos, mass, eps, prm, R, active_idx=act, a_old=None)
    assert np.array_equal(S, oinfo["splitters"])
    got = np.zeros((n, 3)); gp = np.zeros(n); seen = np.zeros(n, bool)
    for r in range(R):
        g = doms[r].gid[doms[r].active.long()].numpy()
        got[g] = res[r][0].numpy(); gp[g] = res[r][1].numpy(); seen[g] = True
    assert np.array_equal(np.flatnonzero(seen), act)
    assert np.abs(got[act] - a_ref).max() <= 1e-5 * np.abs(a_ref).max()
    assert np.abs(gp[act] - p_ref).max() <= 1e-5 * np.abs(p_ref).max()
    assert sum(info["n_exported"].values()) == int(oinfo["n_exported"].sum()) > 0
