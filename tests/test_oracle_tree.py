"""Pins P9..P12, P15 for the oracle's keys / sort / canonical octree / upward pass.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_2606_17145_b200 import workloads as W


def _magic_interleave(q):
    """Magic-mask 21-bit -> every-third-bit spread (independent of the oracle's bit loop)."""
    x = np.asarray(q, dtype=np.uint64) & np.uint64(0x1FFFFF)
    x = (x | (x << np.uint64(32))) & np.uint64(0x1F00000000FFFF)
    x = (x | (x << np.uint64(16))) & np.uint64(0x1F0000FF0000FF)
    x = (x | (x << np.uint64(8))) & np.uint64(0x100F00F00F00F00F)
    x = (x | (x << np.uint64(4))) & np.uint64(0x10C30C30C30C30C3)
    x = (x | (x << np.uint64(2))) & np.uint64(0x1249249249249249)
    return x


def _numpy_keys(pos, L):
    S = np.float32(2097152.0 / float(L))
    t = pos.astype(np.float32) * S                     # one binary32 multiply per axis
    t = np.where(t >= 0, t, np.float32(0))
    t = np.minimum(t, np.float32(2097151.0))
    q = t.astype(np.uint32)
    return (_magic_interleave(q[:, 0]) << np.uint64(2)) | (_magic_interleave(q[:, 1]) << np.uint64(1)) \
        | _magic_interleave(q[:, 2])


def test_p11_interleave_roundtrip_and_magic_masks():
    rng = np.random.default_rng(1)
    qs = rng.integers(0, 1 << 21, size=(2000, 3), dtype=np.uint32)
    qs = np.vstack([qs, [[0, 0, 0], [2097151, 2097151, 2097151], [2097151, 0, 0], [0, 2097151, 0],
                         [0, 0, 2097151], [1, 2, 4], [1 << 20, 0, 1]]]).astype(np.uint32)
    for qx, qy, qz in qs[:300]:
        k = oracle.interleave(qx, qy, qz)
        assert k < (1 << 63)
        assert oracle.deinterleave(k) == (qx, qy, qz)
    mk = (_magic_interleave(qs[:, 0]) << np.uint64(2)) | (_magic_interleave(qs[:, 1]) << np.uint64(1)) \
        | _magic_interleave(qs[:, 2])
    ok = np.array([oracle.interleave(*q) for q in qs], dtype=np.uint64)
    assert np.array_equal(mk, ok)
    # bit placement: x -> 3b+2, y -> 3b+1, z -> 3b
    assert oracle.interleave(1, 0, 0) == 4 and oracle.interleave(0, 1, 0) == 2 and oracle.interleave(0, 0, 1) == 1
    assert oracle.interleave(1 << 20, 0, 0) == 1 << 62


@pytest.mark.parametrize("L", [1.0, 100.0, 400.0])
def test_p11_keys_equal_numpy_float32_keys(L):
    rng = np.random.default_rng(7)
    pos = (rng.random((50000, 3)) * L).astype(np.float32)
    pos[pos >= np.float32(L)] = 0
    pos[:4] = [[0, 0, 0], [np.nextafter(np.float32(L), np.float32(0))] * 3, [L / 2] * 3, [L / 3, 0, L / 7]]
    assert np.array_equal(oracle.keys(pos, L), _numpy_keys(pos, L))


def test_p11_key_scale_facts():
    """L = 1 -> S = 2^21 exactly; L = 100 -> S = 20971.51953125 and the largest
    fp32 below 100 hits the clamp."""
    assert np.float32(2097152.0 / 1.0) == 2097152.0
    assert float(np.float32(2097152.0 / 100.0)) == 20971.51953125
    x = np.nextafter(np.float32(100.0), np.float32(0))
    k = oracle.keys(np.array([[x, x, x]], np.float32), 100.0)[0]
    assert oracle.deinterleave(k) == (2097151, 2097151, 2097151)
    # out-of-range and NaN positions clamp instead of wrapping (R2)
    k = oracle.keys(np.array([[-1.0, np.nan, 1e9]], np.float32), 100.0)[0]
    assert oracle.deinterleave(k) == (0, 0, 2097151)


def test_p11_sorted_keys_follow_octant_paths():
    w = W.uniform_box(8)
    k = oracle.keys(w.pos, w.L)
    perm, ks = oracle.sort(k)
    paths = [tuple(int((int(x) >> (60 - 3 * l)) & 7) for l in range(21)) for x in ks]
    assert paths == sorted(paths)


def test_p12_sort_is_stable_argsort():
    rng = np.random.default_rng(3)
    # many duplicate keys: 1e5 points on a 16^3 grid
    g = rng.integers(0, 16, size=(100000, 3)).astype(np.float32) / 16 + np.float32(1 / 32)
    k = oracle.keys(g, 1.0)
    assert np.unique(k).size <= 4096
    perm, ks = oracle.sort(k)
    ref = np.argsort(k, kind="stable")
    assert np.array_equal(perm, ref.astype(np.uint32))
    assert np.array_equal(ks, k[ref])
    w = W.nfw_box(24, 10)
    k = oracle.keys(w.pos, w.L)
    perm, ks = oracle.sort(k)
    assert np.array_equal(perm, np.argsort(k, kind="stable").astype(np.uint32))


# ---- P10: tree by naive definition (recursive point insertion into cubes) ---------------
def _naive_tree(q, leaf_max):
    """q: integer cell coordinates [N][3] (21 bits) in ORIGINAL order.  Builds the octree by
    recursive splitting of cubes on the point set (no keys, no sorting), then renumbers
    canonically (BFS, children by ascending octant).  Returns the per-node (level, sorted ids)."""
    root = (0, np.arange(q.shape[0]))
    nodes = [root]
    out = []
    j = 0
    while j < len(nodes):
        lv, ids = nodes[j]
        kids = []
        if ids.size > leaf_max and lv < 21:
            b = 20 - lv
            octant = (((q[ids, 0] >> b) & 1) << 2) | (((q[ids, 1] >> b) & 1) << 1) | ((q[ids, 2] >> b) & 1)
            for o in range(8):
                sub = ids[octant == o]
                if sub.size:
                    kids.append((lv + 1, sub))
        out.append((lv, ids, len(nodes) if kids else 0, len(kids)))
        nodes.extend(kids)
        j += 1
    return out


@pytest.mark.parametrize("case", ["uniform", "clustered", "duplicates"])
@pytest.mark.parametrize("leaf_max", [1, 8])
def test_p10_tree_equals_naive_insertion(case, leaf_max):
    rng = np.random.default_rng(11)
    if case == "uniform":
        pos = rng.random((3000, 3)).astype(np.float32)
    elif case == "clustered":
        pos = np.mod(0.5 + 0.01 * rng.standard_normal((3000, 3)) ** 3, 1.0).astype(np.float32)
    else:
        base = rng.random((40, 3)).astype(np.float32)
        pos = base[rng.integers(0, 40, 1500)]            # coincident points -> level-21 leaves
        pos[:200] = np.float32(0.123)
    S = np.float32(2097152.0)
    q = np.minimum((pos * S), np.float32(2097151)).astype(np.int64)
    k = oracle.keys(pos, 1.0)
    perm, ks = oracle.sort(k)
    level, first, count, first_child, n_child = oracle.tree_topology(ks, leaf_max)
    naive = _naive_tree(q, leaf_max)
    assert len(naive) == level.shape[0]
    for j, (lv, ids, fc, nc) in enumerate(naive):
        assert lv == level[j] and ids.size == count[j] and nc == n_child[j] and fc == first_child[j]
        got = np.sort(perm[first[j]:first[j] + count[j]])
        assert np.array_equal(got, np.sort(ids).astype(np.uint32))
    if case == "duplicates":
        assert level.max() == 21


@pytest.mark.parametrize("name", ["uniform32", "nfw256", "zoom"])
def test_p9_tree_invariants(name):
    w = W.make(name, small=True)
    prm = oracle.make_params(w.L, w.r_s)
    t = oracle.build_tree(w.pos, w.mass, w.eps, prm)
    nn, lm = t.n_nodes, 8
    leaf = t.n_child == 0
    assert t.level[0] == 0 and t.first[0] == 0 and t.count[0] == w.n
    assert int(t.count[leaf].sum()) == w.n
    assert np.all((t.count[leaf] <= lm) | (t.level[leaf] == 21))
    assert np.all(t.count[~leaf] > lm)
    assert np.all(np.diff(t.level.astype(int)) >= 0)                     # BFS order
    for j in np.flatnonzero(~leaf):
        ch = np.arange(t.first_child[j], t.first_child[j] + t.n_child[j])
        assert np.all(t.level[ch] == t.level[j] + 1)
        assert t.first[ch[0]] == t.first[j]
        assert np.array_equal(t.first[ch][1:], (t.first[ch] + t.count[ch])[:-1])
        assert t.first[ch[-1]] + t.count[ch[-1]] == t.first[j] + t.count[j]
        assert np.all(t.hmax[ch] <= t.hmax[j])
        # children in ascending octant order, all inside the parent's key prefix
        sh = 60 - 3 * int(t.level[j])
        digs = (t.keys_sorted[t.first[ch]] >> np.uint64(sh)) & np.uint64(7)
        assert np.all(np.diff(digs.astype(int)) > 0)
    # children blocks are contiguous and cover 1..nn-1 exactly once
    fc = t.first_child[~leaf].astype(np.int64)
    nc = t.n_child[~leaf].astype(np.int64)
    assert fc[0] == 1 and np.array_equal(fc[1:], (fc + nc)[:-1]) and fc[-1] + nc[-1] == nn
    # moments
    m64 = w.mass.astype(np.float64)
    assert t.M64[0] == pytest.approx(m64.sum(), rel=1e-12)
    com = (m64[:, None] * w.pos.astype(np.float64)).sum(0) / m64.sum()
    assert np.allclose(t.s64[0], com, rtol=1e-11, atol=0)
    assert np.all(t.lo <= t.s + 1e-6 * w.L) and np.all(t.s <= t.hi + 1e-6 * w.L)
    assert np.all(t.lo[0] == w.pos.min(0)) and np.all(t.hi[0] == w.pos.max(0))
    # AABB inside the cell cube (+- 2 ulp of L); l = L / 2^level exactly
    assert np.array_equal(t.l, (np.float64(w.L) / 2.0 ** t.level.astype(np.float64)).astype(np.float32))
    tol = 4 * np.spacing(np.float32(w.L))
    assert np.all(t.lo >= t.c - 0.5 * t.l[:, None] - tol)
    assert np.all(t.hi <= t.c + 0.5 * t.l[:, None] + tol)
    assert np.array_equal(t.sh, (2.8 * w.eps[t.perm].astype(np.float64)).astype(np.float32))
    assert t.hmax[0] == t.sh.max()


def test_p9_node_records_are_fp32_roundings():
    w = W.make("nfw256", small=True)
    t = oracle.build_tree(w.pos, w.mass, w.eps, oracle.make_params(w.L, w.r_s))
    assert np.array_equal(t.M, t.M64.astype(np.float32))
    assert np.array_equal(t.s, t.s64.astype(np.float32))
    # independent recomputation of a few node moments straight from the particle set
    rng = np.random.default_rng(0)
    for j in rng.integers(0, t.n_nodes, 50):
        sl = slice(int(t.first[j]), int(t.first[j] + t.count[j]))
        m = t.smass[sl].astype(np.float64)
        assert t.M64[j] == pytest.approx(m.sum(), rel=1e-13)
        assert np.allclose(t.s64[j], (m[:, None] * t.spos[sl].astype(np.float64)).sum(0) / m.sum(),
                           rtol=1e-12, atol=0)
        assert np.array_equal(t.lo[j], t.spos[sl].min(0)) and np.array_equal(t.hi[j], t.spos[sl].max(0))


def test_p15_counter_identities():
    w = W.make("nfw256", small=True)
    prm = oracle.make_params(w.L, w.r_s)
    t = oracle.build_tree(w.pos, w.mass, w.eps, prm)
    idx = np.arange(0, w.n, 7, dtype=np.uint32)
    acc, pot, c = oracle.walk(t, idx)                     # geometric
    a_old = np.linalg.norm(acc, axis=1).astype(np.float32)
    for ao in (None, a_old, np.zeros_like(a_old)):
        acc, pot, c = oracle.walk(t, idx, ao)
        c = c.astype(np.int64)
        V_full, V_cull, A_in, A_out, P_in, P_out, P_soft, O_int, O_leaf, C_open, L_open, own = c.T
        assert np.all(V_full + V_cull == 1 + C_open)
        assert np.all(A_in + A_out + O_int + O_leaf == V_full)
        assert np.all(P_in + P_out == L_open - own)
        assert np.all(P_soft <= P_in) and np.all(own <= 1)
        assert np.all(O_int >= 1)                         # the root is always opened (R15)
    # a_old = 0 opens everything: the own leaf is always reached
    assert np.all(own == 1) and np.all(A_in + A_out == 0)
