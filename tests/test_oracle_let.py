"""Pins for row f4 on the oracle side (oracle.walk_ext / direct_ext, oracle/let.py).  CPU only.  References: linearity of
the direct sum over disjoint source sets, the one-domain case = the plain walk, the export filter dropping exactly
nothing, convergence of the domain-decomposed tree force to the global direct sum, a hand-built histogram for the
splitter rule, a closed-form monopole for an external target."""
import numpy as np
import pytest

import oracle
from oracle import let
from paper_2606_17145_b200 import workloads as W


def _small(n_side=12, seed=3, r_s=None):
    w = W.nfw_box(n_side, 6, 100.0, W.SEED0 + seed, name="let_small")
    return w, oracle.make_params(w.L, w.r_s if r_s is None else r_s, alpha=w.alpha, theta=w.theta, leaf_max=8)


def test_direct_sum_is_additive_over_domains():
    """sum over domains of (direct among own particles + direct_ext from the others) = the global direct sum."""
    w, prm = _small()
    own, _ = let.owners(oracle.keys(w.pos, w.L), 3)
    a_ref, p_ref = oracle.direct(w.pos, w.mass, w.eps, prm)
    a, p = np.zeros_like(a_ref), np.zeros_like(p_ref)
    for d in range(3):
        m = np.flatnonzero(own == d)
        o = np.flatnonzero(own != d)
        ad, pd = oracle.direct(w.pos[m], w.mass[m], w.eps[m], prm)
        a[m] += ad
        p[m] += pd
        ae, pe = oracle.direct_ext(w.pos[m], w.mass[m], w.eps[m], prm, w.pos[o], w.eps[o])
        a[o] += ae
        p[o] += pe
    assert np.abs(a - a_ref).max() <= 1e-12 * np.abs(a_ref).max()
    assert np.abs(p - p_ref).max() <= 1e-12 * np.abs(p_ref).max()


def test_one_domain_is_the_plain_walk_bit_for_bit():
    w, prm = _small()
    t = oracle.build_tree(w.pos, w.mass, w.eps, prm)
    a0, p0, _ = oracle.walk(t, None, None, want_counters=False)
    a1, p1, info = let.let_walk(w.pos, w.mass, w.eps, prm, 1)
    assert np.array_equal(a0, a1) and np.array_equal(p0, p1)
    assert np.all(info["owner"] == 0)


def test_external_walk_converges_to_external_direct_sum_and_far_monopole():
    w, prm = _small()
    rng = np.random.default_rng(1)
    t = oracle.build_tree(w.pos, w.mass, w.eps, prm)
    tpos = (rng.random((200, 3)) * w.L).astype(np.float32)
    teps = np.full(200, float(w.eps[0]), np.float32)
    th = oracle.particle_h(teps)
    a_d, p_d = oracle.direct_ext(w.pos, w.mass, w.eps, prm, tpos, teps)
    big = np.full(200, 1e30, np.float32)                    # alpha a_old huge -> everything that may be accepted is
    tiny = np.full(200, 1e-30, np.float32)                  # alpha a_old -> 0: every node is opened
    a_o, p_o, _ = oracle.walk_ext(t, tpos, th, tiny)
    sel = np.linalg.norm(a_d, axis=1) > 0
    assert np.abs(a_o - a_d)[sel].max() <= 1e-11 * np.abs(a_d).max()
    assert np.abs(p_o - p_d).max() <= 1e-11 * np.abs(p_d).max()
    e = []
    for th_ in (0.9, 0.45, 0.2):
        prm2 = oracle.make_params(w.L, prm.r_s, alpha=w.alpha, theta=th_, leaf_max=8)
        a_g, _, _ = oracle.walk_ext(t, tpos, th, None, params=prm2)
        e.append(np.median(np.linalg.norm(a_g - a_d, axis=1)[sel] / np.linalg.norm(a_d, axis=1)[sel]))
    # (slow: a node accepted near r_cut is cut as a whole, R17; the exact limit is the a_old -> 0 case above)
    assert e[0] > e[1] > e[2] and e[2] < 0.5 * e[0]
    # closed form: a tight clump of equal masses and one external target 2.5 r_s away, criterion accepts everything
    c = np.array([50.0, 50.0, 50.0])
    clump = (c + rng.standard_normal((64, 3)) * 1e-4).astype(np.float32)
    cm = np.full(64, 0.25, np.float32)
    prm = oracle.make_params(w.L, 2.0, alpha=w.alpha, theta=w.theta, leaf_max=8)
    tc = oracle.build_tree(clump, cm, np.full(64, 1e-6, np.float32), prm)
    r = 2.5 * prm.r_s
    x = (c + np.array([r, 0, 0])).astype(np.float32)[None]
    a, p, _ = oracle.walk_ext(tc, x, np.array([1e-5], np.float32), big[:1])
    com = clump.astype(np.float64).mean(0)
    d = com - x[0].astype(np.float64)
    rr = np.linalg.norm(d)
    wv = rr / (2 * prm.r_s)
    assert np.allclose(a[0], 16.0 * oracle.split_T(wv) * d / rr ** 3, rtol=1e-6, atol=1e-6 * np.abs(a[0]).max())   # (the node record is fp32, R9)
    assert np.isclose(p[0], -16.0 * oracle.split_E(wv) / rr, rtol=1e-6)


def test_export_filter_drops_exactly_nothing_and_really_filters():
    w, prm = _small(20, 5, r_s=2.0)                           # r_cut = 9 in a box of 100: domains out of reach exist
    rng = np.random.default_rng(2)
    a_old = (rng.random(w.n) * 0.01 + 1e-4).astype(np.float32)
    for R in (3, 8):
        a0, p0, i0 = let.let_walk(w.pos, w.mass, w.eps, prm, R, a_old=a_old, export_all=True)
        a1, p1, i1 = let.let_walk(w.pos, w.mass, w.eps, prm, R, a_old=a_old)
        assert np.array_equal(a0, a1) and np.array_equal(p0, p1)
        assert i1["n_exported"].sum() < i0["n_exported"].sum()
        assert i1["n_local"].sum() == w.n and i1["n_local"].min() > 0


def test_export_filter_level_follows_r_cut():
    """R52: level-2 top boxes are exact only for r_cut <= 0.05 L.  Hand-built case with r_cut = 0.18 L: domain 0 is two
    clumps in different level-2 cells of one level-1 octant; targets of domain 1 sit 6..9 beyond that octant's face
    (outside its 0.6 l guard box), more than r_cut from either clump's box but 8..11 from the octant's centre of mass.
    With a large a_old the level-1 node is accepted and adds a non-zero monopole: a level-2 filter drops it, the rule's
    level-1 filter does not."""
    rng = np.random.default_rng(11)
    L, r_s = 100.0, 4.0                                           # r_cut = 18 > 0.05 L
    clump = lambda c, m: (np.asarray(c) + rng.uniform(-0.5, 0.5, (m, 3))).astype(np.float32)
    pos = np.concatenate([clump((48.0, 5.0, 25.0), 50), clump((48.0, 45.0, 25.0), 50), clump((57.5, 25.0, 25.0), 100)])
    n = pos.shape[0]
    mass = np.full(n, 1.0, np.float32)
    eps = np.full(n, 0.01, np.float32)
    prm = oracle.make_params(L, r_s, alpha=0.005, theta=0.5, leaf_max=8)
    a_old = np.full(n, 1.0e6, np.float32)                         # every node outside its guards is accepted
    a0, p0, i0 = let.let_walk(pos, mass, eps, prm, 2, a_old=a_old, export_all=True)
    assert list(i0["n_local"]) == [100, 100]                      # the two clumps of the octant are domain 0
    assert let.top_level(18.0, L) == 1 and let.top_level(5.0, L) == 2 and let.top_level(5.0001, L) == 1
    a1, p1, i1 = let.let_walk(pos, mass, eps, prm, 2, a_old=a_old)
    assert np.array_equal(a0, a1) and np.array_equal(p0, p1)      # the rule's filter is exact
    a2, p2, i2 = let.let_walk(pos, mass, eps, prm, 2, a_old=a_old, level=2)
    lost = np.abs(a0 - a2).sum(1) > 0
    assert lost[100:].any() and not lost[:100].any()              # level 2 loses the monopole for targets of domain 1
    assert i2["n_exported"].sum() < i1["n_exported"].sum() <= i0["n_exported"].sum()
    # the small-r_cut side of the rule on a random box: level 2 chosen, exact, and a real filter
    w, prm_s = _small(20, 5, r_s=1.0)                             # r_cut = 4.5 <= 0.05 L
    ao = (rng.random(w.n) * 0.01 + 1e-4).astype(np.float32)
    b0, q0, j0 = let.let_walk(w.pos, w.mass, w.eps, prm_s, 3, a_old=ao, export_all=True)
    b1, q1, j1 = let.let_walk(w.pos, w.mass, w.eps, prm_s, 3, a_old=ao)
    assert np.array_equal(b0, b1) and np.array_equal(q0, q1) and j1["n_exported"].sum() < j0["n_exported"].sum()


def test_domain_decomposed_tree_force_converges_to_the_global_direct_sum():
    w, prm = _small()
    a_ref, p_ref = oracle.direct(w.pos, w.mass, w.eps, prm)
    nrm = np.linalg.norm(a_ref, axis=1)
    sel = nrm > 0
    errs = []
    for alpha in (0.05, 0.005, 0.0005):
        prm2 = oracle.make_params(w.L, prm.r_s, alpha=alpha, theta=w.theta, leaf_max=8)
        a, p, _ = let.let_walk(w.pos, w.mass, w.eps, prm2, 3, a_old=nrm.astype(np.float32))
        errs.append(np.percentile(np.linalg.norm(a - a_ref, axis=1)[sel] / nrm[sel], 99))
    assert errs[0] > errs[1] > errs[2] and errs[1] <= 1e-2 and errs[2] < 0.5 * errs[1], errs     # (R30's gate at alpha = 0.005)
    # active subset, arbitrary order: the same numbers as the full call
    act = np.random.default_rng(7).permutation(w.n)[:333].astype(np.uint32)
    a_s, p_s, _ = let.let_walk(w.pos, w.mass, w.eps, prm, 3, active_idx=act, a_old=nrm.astype(np.float32)[act])
    a_f, p_f, _ = let.let_walk(w.pos, w.mass, w.eps, prm, 3, a_old=nrm.astype(np.float32))
    assert np.array_equal(a_s, a_f[act]) and np.array_equal(p_s, p_f[act])


def test_splitter_rule_on_a_hand_built_histogram():
    h = np.zeros(let.N_CELLS, np.int64)
    h[[3, 10, 11, 500, 32767]] = [4, 1, 5, 6, 4]            # N = 20
    S = let.splitters(h, 4)                                 # wants 5, 10, 15 particles before the boundary
    # before cell 11: 5 particles -> S1 = 11;  before cell 500: 10 -> S2 = 500 (first cell with >= 10 before it is 12)
    assert S[0] == 0 and S[4] == let.N_CELLS
    assert S[1] == 11 and S[2] == 12 and S[3] == 501
    keys = np.repeat(np.array([3, 10, 11, 500, 32767], np.uint64), [4, 1, 5, 6, 4]) << np.uint64(let.KEY_SHIFT)
    own, S2 = let.owners(keys, 4)
    assert np.array_equal(S2, S)
    assert np.array_equal(np.bincount(own, minlength=4), [5, 5, 6, 4])
    # every particle of a cell has one owner; owners ascend along the curve
    assert np.all(np.diff(own) >= 0)
