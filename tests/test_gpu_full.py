"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (all targets active /
the config's active subset, leaf_max = 8, potential on).

north_star's tolerance (p99 <= 1e-4, max <= 1e-2 of the per-target relative acceleration error) is a statement
about EVERY active target, and SURVEY.md Sec. 7.3 item 1 measured that samples hide the decision flips that break
the max bar; so configs 1, 2, 3, 4 and 5B are compared on their FULL active sets: the oracle walks every active
target (geometric pass, then the relative pass with a_old = the oracle's geometric |a| rounded to fp32 for all
targets, R23).  Config 5A (134 M targets, ~2 x 6 core-hours of oracle) is compared on a seeded 2^20-target sample
unless OG_TEST_FULL_5A=1.  The measured p99 / max / counts above 1e-4 are printed and appended to
gpurun_out/full_parity.txt.

Config 5 (512^3, both runs) needs ~25 GB of device memory and ~20 GB of host memory; OG_SKIP_HUGE=1 leaves it out."""
import os
import time

import numpy as np
import pytest

import oracle
from paper_2606_17145_b200 import workloads as W
from gpu_common import check_acc, gpu_params, oracle_params, rel_err, rel_err_scalar, to_dev, u32, u64

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B(cuda_device):
    from paper_2606_17145_b200 import binding
    return binding


def _report(name, what, n_cmp, e_acc, e_pot, seconds):
    line = (f"{name:16s} {what:10s} targets {n_cmp:10d}  acc p50 {np.median(e_acc):.2e} p99 {np.percentile(e_acc, 99):.2e} "
            f"max {e_acc.max():.2e} n(>1e-4) {int((e_acc > 1e-4).sum())}  pot p99 {np.percentile(e_pot, 99):.2e} "
            f"max {e_pot.max():.2e} n(>1e-4) {int((e_pot > 1e-4).sum())}  oracle {seconds:.0f} s")
    print(line)
    try:
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        with open(os.path.join(ROOT, "gpurun_out", "full_parity.txt"), "a") as f:
            f.write(line + "\n")
    except OSError:
        pass


def _full_case(B, name, runs=((None, True, None),)):
    """One workload, one tree on each side, then one or more runs (label, use the config's active subset?, nsample);
    nsample = None: every active target is compared; else a seeded sample of that many active targets."""
    import torch
    w = W.make(name)
    ot = oracle.build_tree(w.pos, w.mass, w.eps, oracle_params(w))
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w))
    assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
    # keys / permutation / topology / node records: bit-exact at full size (R27)
    assert B.og_tree_stats(tree)["n_nodes"] == ot.n_nodes
    assert np.array_equal(u64(B.og_tree_get(tree, B.OG_F_KEYS_SORTED)), ot.keys_sorted)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_PERM)), ot.perm)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_INV_PERM)), ot.inv_perm)
    assert np.array_equal(B.og_tree_get(tree, B.OG_F_NODE_LEVEL).cpu().numpy(), ot.level)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_NODE_FIRST)), ot.first)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_NODE_COUNT)), ot.count)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_NODE_FIRST_CHILD)), ot.first_child)
    assert np.array_equal(B.og_tree_get(tree, B.OG_F_NODE_NCHILD).cpu().numpy(), ot.n_child)
    com = B.og_tree_get(tree, B.OG_F_NODE_COM).cpu().numpy()
    assert np.array_equal(com[:, 3], ot.M) and np.array_equal(com[:, :3], ot.s)
    del com
    cell = B.og_tree_get(tree, B.OG_F_NODE_CELL).cpu().numpy()
    assert np.array_equal(cell[:, :3], ot.c) and np.array_equal(cell[:, 3], ot.l)
    del cell
    lo = B.og_tree_get(tree, B.OG_F_NODE_LO).cpu().numpy()
    assert np.array_equal(lo[:, :3], ot.lo) and np.array_equal(lo[:, 3], ot.hmax)
    del lo
    assert np.array_equal(B.og_tree_get(tree, B.OG_F_NODE_HI).cpu().numpy()[:, :3], ot.hi)
    for label, use_active, nsample in runs:
        _one_run(B, w, ot, tree, label or name, w.active_idx if use_active else None, nsample)
    B.og_tree_free(tree)


def _one_run(B, w, ot, tree, name, act_np, nsample):
    """The walk as bench.py launches it: every active target, geometric pass then relative pass."""
    import torch
    act = None if act_np is None else torch.from_numpy(act_np.view(np.int32)).cuda()
    na = w.n if act_np is None else act_np.shape[0]
    a1, p1 = B.og_shortrange_accel(tree, act, None)
    if nsample is None:
        pick = None
        orig = act_np                                  # None -> all particles in identity order
        n_cmp = na
    else:
        rng = np.random.Generator(np.random.PCG64(W.SEED0 + 77))
        pick = np.sort(rng.choice(na, min(nsample, na), replace=False))
        orig = pick.astype(np.uint32) if act_np is None else act_np[pick]
        n_cmp = pick.shape[0]
    sel = (lambda x: x) if pick is None else (lambda x: x[torch.from_numpy(pick).cuda()])
    t0 = time.time()
    ao1, po1, _ = oracle.walk(ot, orig, None, want_counters=False)
    t_or = time.time() - t0
    e1, _ = rel_err(sel(a1).cpu().numpy(), ao1)
    _report(name, "geometric", n_cmp, e1, rel_err_scalar(sel(p1).cpu().numpy(), po1), t_or)
    check_acc(sel(a1).cpu().numpy(), ao1, what=f"{name} full geometric")
    # relative pass (R23): both sides get the oracle's geometric |a| rounded to fp32 on the compared targets
    # (all of them when nothing is sampled; the other targets of a sampled run keep the GPU's own |a|)
    a_old_s = np.linalg.norm(ao1, axis=1).astype(np.float32)
    del ao1, po1
    if pick is None:
        a_old = torch.from_numpy(a_old_s).cuda()
    else:
        a_old = torch.linalg.vector_norm(a1, dim=1).contiguous()
        a_old[torch.from_numpy(pick).cuda()] = torch.from_numpy(a_old_s).cuda()
    a2, p2 = B.og_shortrange_accel(tree, act, a_old)
    assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
    t0 = time.time()
    ao2, po2, _ = oracle.walk(ot, orig, a_old_s, want_counters=False)
    t_or = time.time() - t0
    e2, _ = rel_err(sel(a2).cpu().numpy(), ao2)
    ep = rel_err_scalar(sel(p2).cpu().numpy(), po2)
    _report(name, "relative", n_cmp, e2, ep, t_or)
    check_acc(sel(a2).cpu().numpy(), ao2, what=f"{name} full relative")
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2
    # properties at any size: finite everywhere, potential negative, results independent of launch order
    assert bool(torch.isfinite(a2).all()) and bool(torch.isfinite(p2).all())
    assert bool((p2 <= 0).all())
    a3, p3 = B.og_shortrange_accel(tree, act, a_old)
    assert torch.equal(a2, a3) and torch.equal(p2, p3), "walk is not run-to-run bit-reproducible"


def test_full_uniform32_and_direct_sum(B):
    """configs[0] in full: tree walk vs oracle walk on all 32768 targets, and vs the O(N^2) direct sum (R30)."""
    import torch
    w = W.make("uniform32")
    ot = oracle.build_tree(w.pos, w.mass, w.eps, oracle_params(w))
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w))
    a1, _ = B.og_shortrange_accel(tree, None, None)
    ao1, _, _ = oracle.walk(ot, None, None, want_counters=False)
    check_acc(a1.cpu().numpy(), ao1, what="uniform32 geometric")
    a_old = np.linalg.norm(ao1, axis=1).astype(np.float32)
    a2, p2 = B.og_shortrange_accel(tree, None, torch.from_numpy(a_old).cuda())
    ao2, po2, _ = oracle.walk(ot, None, a_old, want_counters=False)
    check_acc(a2.cpu().numpy(), ao2, what="uniform32 relative")
    ad, pd = oracle.direct(w.pos, w.mass, w.eps, oracle_params(w))
    check_acc(a2.cpu().numpy(), ad, p99=1e-2, mx=1e-1, what="uniform32 tree vs direct")
    a0, _ = B.og_shortrange_accel(tree, None, torch.zeros(w.n, device="cuda"))
    check_acc(a0.cpu().numpy(), ad, p99=2e-5, mx=1e-3, what="uniform32 walk(a_old=0) vs direct")
    B.og_tree_free(tree)


@pytest.mark.parametrize("name", ["lattice128", "nfw256", "zoom"])
def test_full_active_set(B, name):
    """configs 2, 3, 4: every active target against the oracle."""
    _full_case(B, name)


@pytest.mark.skipif(os.environ.get("OG_SKIP_HUGE") == "1", reason="512^3 left out by OG_SKIP_HUGE=1")
def test_nfw512_both_runs(B):
    """config 5 (one 134 M-particle box, one tree): run B = all 13.4 M targets of the seeded 10 % active subset against
    the oracle; run A (all 134 M active) on a seeded 2^20-target sample, or in full with OG_TEST_FULL_5A=1 (hours of
    oracle time)."""
    _full_case(B, "nfw512_active10", runs=(("nfw512_active10", True, None),
                                           ("nfw512", False, None if os.environ.get("OG_TEST_FULL_5A") == "1" else 1 << 20)))
