"""-m gpu: parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(all targets active / the config's active subset, leaf_max = 8, potential on), checked on sampled
outputs the oracle computes one by one, plus properties that hold at any size.

Config 5 (512^3, both runs) needs ~25 GB of device memory, ~20 GB of host memory and ~75 s per run
(measured on the B200 box); set OG_SKIP_HUGE=1 to leave it out."""
import os

import numpy as np
import pytest

import oracle
from paper_2606_17145_b200 import workloads as W
from gpu_common import check_acc, gpu_params, oracle_params, rel_err_scalar, to_dev, u32, u64

pytestmark = pytest.mark.gpu

NSAMPLE = 1 << 15


@pytest.fixture(scope="module")
def B(cuda_device):
    from paper_2606_17145_b200 import binding
    return binding


def _full_case(B, name, nsample=NSAMPLE):
    import torch
    w = W.make(name)
    ot = oracle.build_tree(w.pos, w.mass, w.eps, oracle_params(w))
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w))
    assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
    # keys / permutation / topology: bit-exact at full size
    assert B.og_tree_stats(tree)["n_nodes"] == ot.n_nodes
    assert np.array_equal(u64(B.og_tree_get(tree, B.OG_F_KEYS_SORTED)), ot.keys_sorted)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_PERM)), ot.perm)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_NODE_FIRST)), ot.first)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_NODE_COUNT)), ot.count)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_NODE_FIRST_CHILD)), ot.first_child)
    assert np.array_equal(B.og_tree_get(tree, B.OG_F_NODE_NCHILD).cpu().numpy(), ot.n_child)
    assert np.array_equal(B.og_tree_get(tree, B.OG_F_NODE_COM).cpu().numpy()[:, 3], ot.M)
    # the walk as bench.py launches it: every active target, geometric pass then relative pass
    act_np = w.active_idx
    act = None if act_np is None else torch.from_numpy(act_np.view(np.int32)).cuda()
    na = w.n_active
    a1, p1 = B.og_shortrange_accel(tree, act, None)
    # sample of the active targets (positions in the active order), walked by the oracle one by one
    rng = np.random.Generator(np.random.PCG64(W.SEED0 + 77))
    pick = np.sort(rng.choice(na, min(nsample, na), replace=False))
    orig = pick.astype(np.uint32) if act_np is None else act_np[pick]
    ao1, po1, _ = oracle.walk(ot, orig, None, want_counters=False)
    check_acc(a1[pick].cpu().numpy(), ao1, what=f"{name} full geometric")
    # relative pass: a_old for ALL active targets from the GPU geometric pass, but the sampled targets get the
    # oracle's |a| (R23) so that both sides test identical inputs on the compared targets
    a_old = torch.linalg.vector_norm(a1, dim=1).contiguous()
    a_old_s = np.linalg.norm(ao1, axis=1).astype(np.float32)
    a_old[torch.from_numpy(pick).cuda()] = torch.from_numpy(a_old_s).cuda()
    a2, p2 = B.og_shortrange_accel(tree, act, a_old)
    assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
    ao2, po2, _ = oracle.walk(ot, orig, a_old_s, want_counters=False)
    check_acc(a2[pick].cpu().numpy(), ao2, what=f"{name} full relative")
    ep = rel_err_scalar(p2[pick].cpu().numpy(), po2)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2
    # properties at any size: finite everywhere, potential negative, results independent of launch order
    assert bool(torch.isfinite(a2).all()) and bool(torch.isfinite(p2).all())
    assert bool((p2 <= 0).all())
    a3, p3 = B.og_shortrange_accel(tree, act, a_old)
    assert torch.equal(a2, a3) and torch.equal(p2, p3), "walk is not run-to-run bit-reproducible"
    B.og_tree_free(tree)


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
def test_full_size_sampled(B, name):
    _full_case(B, name)


@pytest.mark.skipif(os.environ.get("OG_SKIP_HUGE") == "1", reason="512^3 left out by OG_SKIP_HUGE=1")
@pytest.mark.parametrize("name", ["nfw512", "nfw512_active10"])
def test_full_size_sampled_huge(B, name):
    _full_case(B, name, nsample=1 << 13)
