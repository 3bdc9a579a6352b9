"""-m gpu: element-by-element parity of the CUDA path (through the C ABI) against the oracle on
the same seeded inputs (BASELINE.json north_star: keys / permutation / topology bit-exact;
acceleration p99 <= 1e-4, max <= 1e-2 per target).  Small variants of all five configs --
sizes the oracle finishes in seconds that still span several tiles and a ragged tail."""
import numpy as np
import pytest

import oracle
from paper_2606_17145_b200 import workloads as W
from gpu_common import (check_acc, gpu_params, oracle_params, rel_err_scalar, to_dev, u32, u64)

pytestmark = pytest.mark.gpu

SMALL = ["uniform32", "lattice128", "nfw256", "zoom", "nfw512", "nfw512_active10"]


@pytest.fixture(scope="module")
def B(cuda_device):
    from paper_2606_17145_b200 import binding
    return binding


_cache = {}


def _case(name, leaf_max=8):
    key = (name, leaf_max)
    if key not in _cache:
        w = W.make(name, small=True)
        t = oracle.build_tree(w.pos, w.mass, w.eps, oracle_params(w, leaf_max))
        _cache[key] = (w, t)
    return _cache[key]


# ---- a1: keys -----------------------------------------------------------------------------
@pytest.mark.parametrize("name", SMALL[:5])
def test_a1_keys_bit_exact(B, name):
    import torch
    w, t = _case(name)
    pos, _, _ = to_dev(w)
    keys, idx = B.og_morton_keys(pos, w.L)
    torch.cuda.synchronize()
    assert np.array_equal(u64(keys), t.keys)
    assert np.array_equal(u32(idx), np.arange(w.n, dtype=np.uint32))


@pytest.mark.parametrize("n", [1, 3, 4, 5, 1023, 4097])
def test_a1_keys_ragged_sizes_and_extremes(B, n):
    import torch
    rng = np.random.default_rng(n)
    L = 100.0
    pos = (rng.random((n, 3)) * L).astype(np.float32)
    pos[0] = [0.0, np.nextafter(np.float32(L), np.float32(0)), 0.0]      # clamp path (R2)
    keys, _ = B.og_morton_keys(torch.from_numpy(pos).cuda(), L)
    assert np.array_equal(u64(keys), oracle.keys(pos, L))


# ---- a2: sort -----------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 31, 4096, 4097, 100_003])
def test_a2_radix_sort_stable_bit_exact(B, n):
    import torch
    rng = np.random.default_rng(100 + n)
    k = rng.integers(0, 1 << 63, n, dtype=np.uint64)
    k[rng.random(n) < 0.3] = k[0]                      # many duplicates: stability = index tie-break
    perm_o, ks_o = oracle.sort(k)
    kd = torch.from_numpy(k.view(np.int64)).cuda()
    vd = torch.arange(n, dtype=torch.int32, device="cuda")
    ks, vs = B.og_radix_sort_pairs(kd, vd)
    torch.cuda.synchronize()
    assert np.array_equal(u64(ks), ks_o)
    assert np.array_equal(u32(vs), perm_o)


def test_a2_radix_sort_partial_bits(B):
    import torch
    n = 50_000
    rng = np.random.default_rng(7)
    k = rng.integers(0, 1 << 20, n, dtype=np.uint64)
    kd = torch.from_numpy(k.view(np.int64)).cuda()
    vd = torch.arange(n, dtype=torch.int32, device="cuda")
    ks, vs = B.og_radix_sort_pairs(kd, vd, 0, 20)      # 3 passes -> result in the alternate buffers
    assert np.array_equal(u32(vs), np.argsort(k, kind="stable").astype(np.uint32))


@pytest.mark.parametrize("begin_bit,end_bit", [(0, 20), (3, 13), (5, 6), (40, 63)])
def test_a2_radix_sort_sorts_on_the_stated_bits_only(B, begin_bit, end_bit):
    """og.h: stable sort by the key bits [begin_bit, end_bit): bits above end_bit (and below begin_bit) are random
    here and must not influence the order, also when the range is not a multiple of 8."""
    import torch
    n = 70_001
    rng = np.random.default_rng(11)
    k = rng.integers(0, 1 << 63, n, dtype=np.uint64)
    kd = torch.from_numpy(k.view(np.int64)).cuda()
    vd = torch.arange(n, dtype=torch.int32, device="cuda")
    ks, vs = B.og_radix_sort_pairs(kd, vd, begin_bit, end_bit)
    field = (k >> np.uint64(begin_bit)) & np.uint64((1 << (end_bit - begin_bit)) - 1)
    ref = np.argsort(field, kind="stable").astype(np.uint32)
    assert np.array_equal(u32(vs), ref)
    assert np.array_equal(u64(ks), k[ref])


# ---- a2..a5: permutation, topology, node records -------------------------------------------
@pytest.mark.parametrize("name,leaf_max", [(n, 8) for n in SMALL[:5]] + [("nfw256", 1), ("nfw256", 32)])
def test_tree_bit_exact(B, name, leaf_max):
    w, t = _case(name, leaf_max)
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w, leaf_max, max_nodes=3 * w.n if leaf_max < 4 else 0))
    assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
    st = B.og_tree_stats(tree)
    assert st["n_nodes"] == t.n_nodes
    assert st["max_level"] == int(t.level.max())
    assert np.array_equal(u64(B.og_tree_get(tree, B.OG_F_KEYS_SORTED)), t.keys_sorted)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_PERM)), t.perm)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_INV_PERM)), t.inv_perm)
    assert np.array_equal(B.og_tree_get(tree, B.OG_F_NODE_LEVEL).cpu().numpy(), t.level)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_NODE_FIRST)), t.first)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_NODE_COUNT)), t.count)
    assert np.array_equal(u32(B.og_tree_get(tree, B.OG_F_NODE_FIRST_CHILD)), t.first_child)
    assert np.array_equal(B.og_tree_get(tree, B.OG_F_NODE_NCHILD).cpu().numpy(), t.n_child)
    # sorted copies and h = fl32(2.8 eps) (R9)
    spos = B.og_tree_get(tree, B.OG_F_SPOS).cpu().numpy()
    assert np.array_equal(spos[:, :3], t.spos) and np.array_equal(spos[:, 3], t.smass)
    assert np.array_equal(B.og_tree_get(tree, B.OG_F_SH).cpu().numpy(), t.sh)
    # node records (R9, R27): same fp64 summation order on both sides -> equal fp32 bits
    com = B.og_tree_get(tree, B.OG_F_NODE_COM).cpu().numpy()
    cell = B.og_tree_get(tree, B.OG_F_NODE_CELL).cpu().numpy()
    lo = B.og_tree_get(tree, B.OG_F_NODE_LO).cpu().numpy()
    hi = B.og_tree_get(tree, B.OG_F_NODE_HI).cpu().numpy()
    assert np.array_equal(com[:, 3], t.M)
    assert np.array_equal(com[:, :3], t.s)
    assert np.array_equal(cell[:, :3], t.c) and np.array_equal(cell[:, 3], t.l)
    assert np.array_equal(lo[:, :3], t.lo) and np.array_equal(hi[:, :3], t.hi)
    assert np.array_equal(lo[:, 3], t.hmax)
    B.og_tree_free(tree)


# ---- a6..a7: walk ---------------------------------------------------------------------------
def _walk_case(B, name, leaf_max=8):
    import torch
    w, t = _case(name, leaf_max)
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w, leaf_max, flags=B.OG_COUNT))
    act = None if w.active_idx is None else torch.from_numpy(w.active_idx.view(np.int32)).cuda()
    # pass 1: geometric criterion (theta = 0.5), parity-checked on its own (R23)
    a1, p1 = B.og_shortrange_accel(tree, act, None)
    st1 = B.og_tree_stats(tree)
    ao1, po1, c1 = oracle.walk(t, w.active_idx, None)
    q, m = check_acc(a1.cpu().numpy(), ao1, what=f"{name} geometric")
    ep = rel_err_scalar(p1.cpu().numpy(), po1)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2
    # pass 2: relative criterion with the oracle's |a| rounded to fp32 on both sides (R23)
    a_old = np.linalg.norm(ao1, axis=1).astype(np.float32)
    a2, p2 = B.og_shortrange_accel(tree, act, torch.from_numpy(a_old).cuda())
    st2 = B.og_tree_stats(tree)
    assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
    ao2, po2, c2 = oracle.walk(t, w.active_idx, a_old)
    check_acc(a2.cpu().numpy(), ao2, what=f"{name} relative")
    ep = rel_err_scalar(p2.cpu().numpy(), po2)
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2
    # interaction totals (R27): decisions equal the oracle's -> sums agree to 1e-4 relative
    for st, c in ((st1, c1), (st2, c2)):
        for key, col in (("A_in", 2), ("P_in", 4), ("P_soft", 6)):
            ref = int(c[:, col].sum())
            assert abs(st[key] - ref) <= max(2, 1e-4 * ref), (key, st[key], ref)
    B.og_tree_free(tree)


@pytest.mark.parametrize("name", SMALL)
def test_walk_group_matches_oracle(B, name):
    _walk_case(B, name)


@pytest.mark.parametrize("leaf_max", [1, 32])
def test_walk_other_leaf_sizes(B, leaf_max):
    import torch
    w, t = _case("nfw256", leaf_max)
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w, leaf_max, max_nodes=3 * w.n))
    a1, _ = B.og_shortrange_accel(tree, None, None, want_pot=False)
    ao1, _, _ = oracle.walk(t, None, None, want_counters=False)
    check_acc(a1.cpu().numpy(), ao1, what=f"leaf_max={leaf_max}")
    B.og_tree_free(tree)


def test_config1_against_direct_sum(B):
    """BASELINE.json configs[0]: 'also checked against O(N^2) direct short-range summation' (R30),
    here on the 16^3 variant; the full 32^3 case is in test_gpu_full.py."""
    import torch
    w, t = _case("uniform32")
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w))
    ad, pd = oracle.direct(w.pos, w.mass, w.eps, oracle_params(w))
    a_old = np.linalg.norm(ad, axis=1).astype(np.float32)
    a, p = B.og_shortrange_accel(tree, None, torch.from_numpy(a_old).cuda())
    # tree error itself (alpha = 0.005): R30 gate p99 <= 1e-2
    check_acc(a.cpu().numpy(), ad, p99=1e-2, mx=1e-1, what="tree vs direct")
    # with a_old = 0 the walk IS the direct sum (P8): fp32 rounding only
    a0, p0 = B.og_shortrange_accel(tree, None, torch.zeros(w.n, device="cuda"))
    check_acc(a0.cpu().numpy(), ad, p99=2e-5, mx=1e-3, what="walk(a_old=0) vs direct")
    B.og_tree_free(tree)
