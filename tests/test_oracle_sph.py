"""Pins for oracle/sph.py (row f3: SPH density / smoothing length).  CPU only.  References: kernel
quadrature and identities, closed-form configurations solved with an independent scalar root finder, exact scaling laws."""
import math

import numpy as np
import pytest
from scipy import integrate, optimize

from oracle import sph


def test_kernel_normalisation_continuity_and_values():
    # int W d^3r = 1  <=>  4 pi (8 / pi) int_0^1 w(u) u^2 du = 1
    val, _ = integrate.quad(lambda u: float(sph.w_kernel(u)) * u * u, 0, 1, points=[0.5])
    assert abs(32.0 * val - 1.0) < 1e-12
    assert sph.w_kernel(0.0) == 1.0 and sph.w_kernel(1.0) == 0.0 and sph.w_kernel(1.5) == 0.0
    assert abs(float(sph.w_kernel(0.5)) - 0.25) < 1e-15                       # both branches meet at 1/4
    assert abs(float(sph.w_kernel(0.5 + 1e-9)) - float(sph.w_kernel(0.5 - 1e-9))) < 1e-8
    u = np.linspace(0, 1, 2001)
    assert np.all(np.diff(sph.w_kernel(u)) <= 0)                              # decreasing: N(h) increases with h


@pytest.mark.parametrize("K,r0", [(6, 0.01), (12, 0.02), (40, 0.005)])
def test_shell_of_neighbours_closed_form(K, r0):
    """A target with K neighbours all at the same distance r0 (random directions) in an otherwise empty box:
    N(h) = (32/3) [w(0) + K w(r0 / h)], rho = (8 / (pi h^3)) [m_0 + K m w(r0 / h)].  The root comes from brentq on that
    scalar expression, not from the oracle."""
    rng = np.random.default_rng(K)
    L, n_des = 1.0, 32.0
    d = rng.standard_normal((K, 3))
    d *= r0 / np.linalg.norm(d, axis=1)[:, None]
    pos = np.vstack([[0.5, 0.5, 0.5], 0.5 + d])
    mass = np.concatenate([[2.0], np.full(K, 0.5)])
    if (32.0 / 3.0) * (1 + K) <= n_des:
        pytest.skip("N can never reach n_des")
    f = lambda h: (32.0 / 3.0) * (1.0 + K * float(sph.w_kernel(r0 / h))) - n_des
    h_ref = optimize.brentq(f, r0 * 1.0000001, 100 * r0, xtol=1e-15, rtol=1e-14)
    h, rho, nn = sph.sph_density(pos, mass, L, n_des, targets=[0])
    assert h[0] == pytest.approx(h_ref, rel=1e-10)
    assert nn[0] == pytest.approx(n_des, rel=1e-10)
    assert rho[0] == pytest.approx(8 / (math.pi * h_ref ** 3) * (2.0 + K * 0.5 * float(sph.w_kernel(r0 / h_ref))), rel=1e-9)


def test_root_scaling_laws_and_periodic_images():
    rng = np.random.default_rng(2)
    n, L, n_des = 3000, 1.0, 40.0
    pos = rng.random((n, 3)) * L
    mass = rng.random(n) + 0.5
    t = np.arange(0, n, 37)
    h, rho, nn = sph.sph_density(pos, mass, L, n_des, targets=t)
    assert np.allclose(nn, n_des, rtol=1e-10)
    # lengths x lam: h x lam, rho / lam^3; masses x c: h unchanged, rho x c
    h2, rho2, _ = sph.sph_density(pos * 3.0, mass * 5.0, L * 3.0, n_des, targets=t)
    assert np.allclose(h2, 3.0 * h, rtol=1e-9) and np.allclose(rho2, 5.0 * rho / 27.0, rtol=1e-9)
    # a rigid shift across the periodic wall changes nothing
    h3, rho3, _ = sph.sph_density(np.mod(pos + [0.37, 0.81, 0.05], L), mass, L, n_des, targets=t)
    assert np.allclose(h3, h, rtol=1e-9) and np.allclose(rho3, rho, rtol=1e-9)
    # sanity of the scale: a Poisson field's SPH density sits above the mean by about the self term 1 / sum_j w.  This pins
    # nothing (the pins are the closed forms above); the upper bound was first written as 1.6 and widened to 2.0 before any
    # kernel existed: with n_des = 32 the self term W(0, h) m alone is (32/3) / n_des = 1/3 of the mean, and the
    # constrained-h estimator on a Poisson field adds a comparable bias, so 1.6 left no margin across seeds; no passage of
    # the paper fixes this number.
    assert 1.0 < np.mean(rho) / (mass.sum() / L ** 3) < 2.0


def test_brute_force_neighbour_sum_agrees():
    """The library neighbour search is only a candidate filter: the same N and rho from an O(N) sum over ALL particles."""
    rng = np.random.default_rng(4)
    n, L = 800, 2.0
    pos = rng.random((n, 3)) * L
    mass = rng.random(n)
    t = [0, 13, 799]
    h, rho, nn = sph.sph_density(pos, mass, L, 33.0, targets=t)
    for k, i in enumerate(t):
        d = pos - pos[i]
        d -= L * np.round(d / L)
        r = np.sqrt((d * d).sum(1))
        assert sph.neighbour_number(r, h[k]) == pytest.approx(33.0, rel=1e-10)
        assert sph.density_at(r, mass, h[k]) == pytest.approx(rho[k], rel=1e-12)
