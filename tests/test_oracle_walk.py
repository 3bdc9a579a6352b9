"""Pins P6, P7, P8, P14 (+ an independent brute-force re-walk) for the oracle's walk and
direct sum.  CPU only."""
import math

import numpy as np
import pytest

import oracle
from paper_2606_17145_b200 import workloads as W


def _clustered(n, seed=5, L=1.0):
    rng = np.random.default_rng(seed)
    ctr = rng.random((6, 3)) * L
    pos = ctr[rng.integers(0, 6, n)] + 0.03 * L * rng.standard_normal((n, 3))
    pos = np.mod(pos, L).astype(np.float32)
    pos[pos >= np.float32(L)] = 0
    mass = (rng.random(n) + 0.5).astype(np.float32) / n
    eps = np.full(n, 0.002 * L, np.float32)
    return pos, mass, eps


def test_p6_direct_sum_momentum_conservation():
    pos, mass, eps = _clustered(2000)
    prm = oracle.make_params(1.0, 0.03)
    acc, pot = oracle.direct(pos, mass, eps, prm)
    m = mass.astype(np.float64)
    tot = np.linalg.norm((m[:, None] * acc).sum(0))
    assert tot / (m * np.linalg.norm(acc, axis=1)).sum() <= 1e-13
    # pairwise potential is symmetric: sum_i m_i phi_i = 2 * (pair energy) -> finite, negative
    assert (m * pot).sum() < 0


@pytest.mark.parametrize("n", [8, 16])
def test_p7_perfect_lattice_has_zero_force(n):
    L = 1.0
    g = ((np.arange(n) + 0.5) / n).astype(np.float32)          # exact in fp32
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    N = n ** 3
    mass = np.full(N, 1.0 / N, np.float32)
    eps = np.full(N, 0.02 / n, np.float32)
    prm = oracle.make_params(L, 1.25 / n if n == 16 else 0.1)   # r_cut < L/2
    bound = 1e-12 * (1.0 / N) * n * n
    acc, _ = oracle.direct(pos, mass, eps, prm)
    assert np.linalg.norm(acc, axis=1).max() <= bound
    t = oracle.build_tree(pos, mass, eps, prm)
    acc_w, _, _ = oracle.walk(t, None, np.zeros(N, np.float32))
    assert np.linalg.norm(acc_w, axis=1).max() <= bound


@pytest.mark.parametrize("leaf_max", [1, 4, 8, 32])
def test_p8_walk_with_zero_aold_equals_direct_sum(leaf_max):
    pos, mass, eps = _clustered(3000, seed=9)
    prm = oracle.make_params(1.0, 0.02, leaf_max=leaf_max)
    t = oracle.build_tree(pos, mass, eps, prm)
    acc_w, pot_w, cnt = oracle.walk(t, None, np.zeros(3000, np.float32))
    acc_d, pot_d = oracle.direct(pos, mass, eps, prm)
    scale = np.linalg.norm(acc_d, axis=1).max()
    assert np.abs(acc_w - acc_d).max() <= 1e-12 * scale
    assert np.abs(pot_w - pot_d).max() <= 1e-12 * np.abs(pot_d).max()
    assert np.all(cnt[:, 2] == 0)                                # nothing accepted as a node


def test_p8_tree_error_decreases_with_alpha():
    pos, mass, eps = _clustered(4096, seed=13)
    prm0 = oracle.make_params(1.0, 0.03)
    acc_d, _ = oracle.direct(pos, mass, eps, prm0)
    t = oracle.build_tree(pos, mass, eps, prm0)
    a_old = np.linalg.norm(acc_d, axis=1).astype(np.float32)
    med = []
    for alpha in (1e-1, 1e-2, 1e-3, 1e-4, 1e-5, 1e-6):
        prm = oracle.make_params(1.0, 0.03, alpha=alpha)
        acc, _, _ = oracle.walk(t, None, a_old, params=prm)
        e = np.linalg.norm(acc - acc_d, axis=1) / np.linalg.norm(acc_d, axis=1)
        med.append(np.mean(e))
    assert all(b <= a for a, b in zip(med, med[1:])), med
    assert med[0] > 1e-4 and med[-1] < 1e-7


def test_p8_geometric_theta_converges_too():
    pos, mass, eps = _clustered(2048, seed=17)
    acc_d, _ = oracle.direct(pos, mass, eps, oracle.make_params(1.0, 0.03))
    errs = []
    for theta in (1.0, 0.5, 0.25, 0.05):
        prm = oracle.make_params(1.0, 0.03, theta=theta)
        t = oracle.build_tree(pos, mass, eps, prm)
        acc, _, _ = oracle.walk(t)
        errs.append(np.mean(np.linalg.norm(acc - acc_d, axis=1) / np.linalg.norm(acc_d, axis=1)))
    assert all(b <= a for a, b in zip(errs, errs[1:])), errs
    assert errs[-1] < 1e-6


def test_p14_newtonian_special_case_is_plain_numpy_sum():
    """r_s huge (r_cut just under L/2), eps -> 0: the direct sum is a plain Newtonian
    nearest-image sum restricted to r < r_cut with T, E -> 1 for r << r_s."""
    rng = np.random.default_rng(2)
    n, L = 300, 1.0
    pos = (0.5 + 0.002 * rng.standard_normal((n, 3))).astype(np.float32)   # r ~ 1e-2 << r_s
    mass = (rng.random(n) + 0.5).astype(np.float32)
    eps = np.full(n, 1e-12, np.float32)
    rs = L / 9.1
    acc, pot = oracle.direct(pos, mass, eps, oracle.make_params(L, rs))
    p = pos.astype(np.float64)
    d = p[None, :, :] - p[:, None, :]
    d -= L * np.round(d / L)
    r = np.linalg.norm(d, axis=2)
    np.fill_diagonal(r, 1.0)                     # d = 0 on the diagonal: no self term
    w = r / (2 * rs)
    c3 = 4 / (3 * math.sqrt(math.pi))
    Tser = 1 - c3 * w ** 3 + (2 / (5 * math.sqrt(math.pi))) * 2 * w ** 5     # 1 - 4w^3/(3 sqrt pi) + 4 w^5/(5 sqrt pi)
    a_ref = (mass[None, :, None] * d * (Tser / r ** 3)[:, :, None]).sum(1)
    assert np.linalg.norm(acc - a_ref, axis=1).max() <= 1e-9 * np.linalg.norm(a_ref, axis=1).max()


def test_walk_matches_independent_python_walk():
    """Re-walk a few targets with a separate pure-Python/numpy implementation of C6 that reads
    only the tree arrays (a dropped guard, a wrong sign or a transposed operand in oracle.c
    shows up here)."""
    w = W.nfw_box(20, 6, L=100.0)
    prm = oracle.make_params(w.L, w.r_s)
    t = oracle.build_tree(w.pos, w.mass, w.eps, prm)
    acc_g, _, _ = oracle.walk(t)
    a_old = np.linalg.norm(acc_g, axis=1).astype(np.float32)
    acc_o, pot_o, cnt = oracle.walk(t, None, a_old)
    L = float(np.float32(w.L)); rs = float(np.float32(w.r_s)); rc = 4.5 * rs
    alpha = float(np.float32(0.005))
    sp = t.spos.astype(np.float64); sm = t.smass.astype(np.float64); sh = t.sh.astype(np.float64)

    def wrap(d):
        return d - L * np.round(d / L)

    def Tf(x):
        return math.erfc(x) + 2 * x / math.sqrt(math.pi) * math.exp(-x * x)

    def walk_one(i):
        slot = int(t.inv_perm[i]); x = sp[slot]; hi_ = sh[slot]; A = alpha * float(a_old[i])
        acc = np.zeros(3); pot = 0.0
        stack = [0]
        while stack:
            n = stack.pop()
            lo, hi = t.lo[n].astype(float), t.hi[n].astype(float)
            e = np.maximum(np.abs(wrap(x - 0.5 * (lo + hi))) - 0.5 * (hi - lo), 0)
            if np.any(e > rc):
                continue
            d = wrap(t.s[n].astype(float) - x); r2 = d @ d
            M, l = float(t.M[n]), float(t.l[n])
            op = M * l * l > A * r2 * r2
            op |= bool(np.all(np.abs(wrap(t.c[n].astype(float) - x)) < 0.6 * l))
            op |= r2 < max(hi_, float(t.hmax[n])) ** 2
            if not op:
                r = math.sqrt(r2)
                if r < rc:
                    acc += M * d * Tf(r / (2 * rs)) / r ** 3
                    pot -= M * math.erfc(r / (2 * rs)) / r
            elif t.n_child[n] == 0:
                for s in range(int(t.first[n]), int(t.first[n] + t.count[n])):
                    if s == slot:
                        continue
                    dd = wrap(sp[s] - x); r = math.sqrt(dd @ dd)
                    if r < rc:
                        h = max(hi_, sh[s])
                        acc += sm[s] * dd * oracle.spline_g(r, h) * Tf(r / (2 * rs))
                        pot += sm[s] * oracle.spline_p(r, h) * math.erfc(r / (2 * rs))
            else:
                stack.extend(range(int(t.first_child[n]), int(t.first_child[n] + t.n_child[n])))
        return acc, pot

    for i in (0, 1, 777, 4000, w.n - 1):
        a, p = walk_one(i)
        assert np.allclose(a, acc_o[i], rtol=1e-11, atol=0)
        assert p == pytest.approx(pot_o[i], rel=1e-11)


def test_config1_tree_vs_direct_r30():
    """R30: config 1 (32^3 uniform) relative-criterion walk vs O(N^2) direct sum; gate p99 <= 1e-2."""
    w = W.make("uniform32")
    prm = oracle.make_params(w.L, w.r_s)
    t = oracle.build_tree(w.pos, w.mass, w.eps, prm)
    acc_g, _, _ = oracle.walk(t)
    acc, pot, cnt = oracle.walk(t, None, np.linalg.norm(acc_g, axis=1).astype(np.float32))
    idx = np.arange(0, w.n, 8, dtype=np.uint32)
    acc_d, pot_d = oracle.direct(w.pos, w.mass, w.eps, prm, idx)
    e = np.linalg.norm(acc[idx] - acc_d, axis=1) / np.linalg.norm(acc_d, axis=1)
    assert np.percentile(e, 99) <= 1e-2 and np.median(e) <= 1e-6
