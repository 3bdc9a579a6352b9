"""Pins P1..P5, P13 for the oracle's pair kernel.  CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate

import oracle
from conftest import golden_rows

H = 0.00175            # 2.8 * 0.02/32
RS = 1.25 / 64
MJ = 1.0 / 32768


def test_p1_spline_golden():
    for u, g, p in golden_rows("spline.txt"):
        u, g, p = float(u), float(g), float(p)
        for h in (1.0, H, 3.7):
            assert oracle.spline_g(u * h, h) * h ** 3 == pytest.approx(g, rel=1e-12)
            assert oracle.spline_p(u * h, h) * h == pytest.approx(p, rel=1e-12)


def test_p1_spline_identities_and_continuity():
    h = 0.37
    assert oracle.spline_g(0.5 * h, h) * h ** 3 == pytest.approx(76 / 15, rel=1e-13)
    assert oracle.spline_p(0.5 * h, h) * h == pytest.approx(-28 / 15, rel=1e-13)
    assert oracle.spline_g(0.0, h) * h ** 3 == pytest.approx(32 / 3, rel=1e-13)
    assert oracle.spline_p(0.0, h) * h == pytest.approx(-14 / 5, rel=1e-13)
    for u0 in (0.5, 1.0):
        for f in (oracle.spline_g, oracle.spline_p):
            a, b = f((u0 - 1e-9) * h, h), f((u0 + 1e-9) * h, h)
            assert a == pytest.approx(b, rel=1e-7)
    # Newtonian outside h
    assert oracle.spline_g(2 * h, h) == pytest.approx(1 / (2 * h) ** 3, rel=1e-15)
    assert oracle.spline_p(2 * h, h) == pytest.approx(-1 / (2 * h), rel=1e-15)


def _W(u):
    """Gadget-2 cubic-spline density kernel, unit mass, h = 1."""
    if u < 0.5:
        return 8 / math.pi * (1 - 6 * u * u + 6 * u ** 3)
    if u < 1:
        return 8 / math.pi * 2 * (1 - u) ** 3
    return 0.0


def test_p1_spline_is_enclosed_mass_of_density_kernel():
    """g(r) = M_enc(r)/r^3 and p(r) = -(M_enc/r + int_r^1 4 pi u W du) by quadrature of W."""
    for u in (0.1, 0.25, 0.4, 0.5, 0.6, 0.75, 0.9, 0.999):
        pts = [x for x in (0.5,) if x < u]
        menc = integrate.quad(lambda t: 4 * math.pi * t * t * _W(t), 0, u, points=pts or None,
                              epsabs=1e-13, epsrel=1e-12)[0]
        pts2 = [x for x in (0.5,) if u < x]
        outer = integrate.quad(lambda t: 4 * math.pi * t * _W(t), u, 1, points=pts2 or None,
                               epsabs=1e-13, epsrel=1e-12)[0]
        assert oracle.spline_g(u, 1.0) == pytest.approx(menc / u ** 3, rel=1e-11)
        assert oracle.spline_p(u, 1.0) == pytest.approx(-(menc / u + outer), rel=1e-11)


def test_p2_split_factor_golden_and_mpmath():
    mp.mp.dps = 40
    for kind, w, v in golden_rows("split_factor.txt"):
        w, v = float(w), float(v)
        got = oracle.split_T(w) if kind == "T" else oracle.split_E(w)
        assert got == pytest.approx(v, rel=2e-13, abs=1e-15)
    for w in np.linspace(0.0, 2.3, 47):
        ref = mp.erfc(w) + 2 * mp.mpf(float(w)) / mp.sqrt(mp.pi) * mp.exp(-mp.mpf(float(w)) ** 2)
        assert oracle.split_T(w) == pytest.approx(float(ref), rel=1e-14)
        assert oracle.split_E(w) == pytest.approx(float(mp.erfc(float(w))), rel=1e-13)


def test_p2_split_series_and_derivative():
    c3 = 4 / (3 * math.sqrt(math.pi))
    assert c3 == pytest.approx(0.752252778063675, rel=1e-14)
    for w in (1e-3, 1e-2, 3e-2):
        # T = 1 - c3 w^3 + (2/(5 sqrt(pi))) ... : next term is O(w^5)
        assert oracle.split_T(w) - (1 - c3 * w ** 3) == pytest.approx(0.0, abs=2 * w ** 5)
    for w in (0.2, 0.7, 1.3, 2.1):
        dw = 1e-5
        num = (oracle.split_T(w + dw) - oracle.split_T(w - dw)) / (2 * dw)
        assert num == pytest.approx(-(4 * w * w / math.sqrt(math.pi)) * math.exp(-w * w), rel=1e-8)


def _r_of(expr):
    if expr.endswith("rs"):
        return float(expr[:-2]) * RS
    return float(expr[:-1]) * H


@pytest.mark.parametrize("placement", ["plain", "wall", "oblique", "oblique_wall"])
def test_p3_two_particle_closed_form(placement):
    prm = oracle.make_params(1.0, RS)
    for expr, amag, phi in golden_rows("two_particle.txt"):
        r, amag, phi = _r_of(expr), float(amag), float(phi)
        if placement == "plain":
            x1 = np.array([0.3, 0.4, 0.6]); x2 = x1 + np.array([r, 0, 0])
        elif placement == "wall":
            x1 = np.array([1.0 - r / 2, 0.4, 0.6]); x2 = np.array([r / 2, 0.4, 0.6])
        elif placement == "oblique":
            n = np.array([1.0, -2.0, 2.0]) / 3.0
            x1 = np.array([0.5, 0.5, 0.5]); x2 = x1 + r * n
        else:
            n = np.array([2.0, 3.0, -6.0]) / 7.0
            x1 = np.array([0.999999, 1e-7, 0.99999]); x2 = np.mod(x1 + r * n, 1.0)
            n = n  # direction from 1 to 2 through the wall
        kind, acc, pot = oracle.pair_eval(prm, x1, H, x2, MJ, H)
        assert np.linalg.norm(acc) == pytest.approx(amag, rel=1e-9 if "wall" in placement else 1e-12,
                                                    abs=0)
        assert pot == pytest.approx(phi, rel=1e-9 if "wall" in placement else 1e-12, abs=0)
        if amag > 0:
            # force on 1 points to 2
            d = x2 - x1
            d -= np.round(d)
            assert np.dot(acc, d) > 0
            assert np.linalg.norm(np.cross(acc, d)) <= 1e-9 * np.linalg.norm(acc) * np.linalg.norm(d)
            # Newton's third law: m1 a1 = -m2 a2
            _, acc2, _ = oracle.pair_eval(prm, x2, H, x1, MJ, H)
            assert np.allclose(acc, -acc2, rtol=1e-12, atol=0)


def test_p4_zero_beyond_rcut_exact():
    prm = oracle.make_params(1.0, RS)
    rcut = 4.5 * RS
    x1 = np.array([0.25, 0.25, 0.25])
    for r in (rcut, rcut * (1 + 1e-15), rcut * 1.0001, 2 * rcut, 0.49):
        kind, acc, pot = oracle.pair_eval(prm, x1, H, x1 + np.array([r, 0, 0]), MJ, H)
        assert kind == 0 and pot == 0.0 and np.all(acc == 0.0)
    kind, acc, pot = oracle.pair_eval(prm, x1, H, x1 + np.array([rcut * (1 - 1e-12), 0, 0]), MJ, H)
    assert kind == 1 and acc[0] > 0 and pot < 0


def test_p3_coincident_and_unequal_softening():
    prm = oracle.make_params(1.0, RS)
    x = np.array([0.5, 0.5, 0.5])
    kind, acc, pot = oracle.pair_eval(prm, x, H, x, MJ, 2 * H)      # r = 0, h = max = 2H (R19)
    assert kind == 2 and np.all(acc == 0.0)
    assert pot == pytest.approx(-(14 / 5) * MJ / (2 * H), rel=1e-14)
    # h = max(h_i, h_j): symmetric in the two softenings
    xj = x + np.array([0.6 * H, 0, 0])
    _, a1, p1 = oracle.pair_eval(prm, x, H, xj, MJ, 2 * H)
    _, a2, p2 = oracle.pair_eval(prm, x, 2 * H, xj, MJ, H)
    assert np.array_equal(a1, a2) and p1 == p2
    w = 0.6 * H / (2 * RS)
    assert a1[0] == pytest.approx(MJ * 0.6 * H * oracle.spline_g(0.6 * H, 2 * H) * oracle.split_T(w),
                                  rel=1e-14)


def test_p5_newtonian_limit():
    """r_s = L/9.1 (r_cut < L/2), r <= 1e-3 r_s, r > h:  |a| r^2/(G m) = 1 - 0.7523 w^3."""
    rs = 1.0 / 9.1
    prm = oracle.make_params(1.0, rs)
    h = 1e-7
    x = np.array([0.5, 0.5, 0.5])
    for r in (1e-3 * rs, 3e-4 * rs, 1e-5 * rs):
        _, acc, pot = oracle.pair_eval(prm, x, h, x + np.array([0, r, 0]), MJ, h)
        w = r / (2 * rs)
        assert acc[1] * r * r / MJ == pytest.approx(1 - 0.752252778063675 * w ** 3, abs=1e-9)


def test_p13_potential_force_consistency():
    """For r >= h the potential is the integral of the force:  d phi/dr = +|a| (phi < 0)."""
    prm = oracle.make_params(1.0, RS)
    x = np.array([0.5, 0.5, 0.5])
    for r in (1.2 * H, 3 * H, 0.5 * RS, RS, 2 * RS, 4 * RS):
        dr = 1e-6 * r
        _, a, _ = oracle.pair_eval(prm, x, H, x + np.array([r, 0, 0]), MJ, H)
        _, _, pp = oracle.pair_eval(prm, x, H, x + np.array([r + dr, 0, 0]), MJ, H)
        _, _, pm = oracle.pair_eval(prm, x, H, x + np.array([r - dr, 0, 0]), MJ, H)
        assert (pp - pm) / (2 * dr) == pytest.approx(a[0], rel=1e-7)
