"""oracle.sph -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain fp64 NumPy restatement of the SPH density / smoothing-length step ("the SPH
density module ... operates as an iterative process, aiming to determine a smoothing length containing a fixed number of
neighbours", :74 "collects all neighbours within a sphere around the target particle").  The paper prints no formula;
readings R43..R47 of DESIGN.md Sec. 12 (Gadget-2's SPH, Springel 2005):

  R43  kernel with compact support h:  W(r, h) = (8 / (pi h^3)) w(r / h),
       w(u) = 1 - 6 u^2 + 6 u^3 (u <= 1/2),  2 (1 - u)^3 (1/2 < u <= 1),  0 (u > 1).
  R44  kernel-weighted neighbour number  N_i(h) = (4 pi / 3) h^3 sum_j W(r_ij, h)  (all particles j, j = i included,
       nearest periodic image).  N_i is continuous and strictly increasing in h once h exceeds 0, so
  R45  the smoothing length h_i is THE ROOT of N_i(h) = N_des: a plain definition, found here by bisection to 1e-13.
  R46  density  rho_i = sum_j m_j W(r_ij, h_i)  with that h_i.
  R47  the iteration by which an implementation reaches the root is free; it stops at |N_i - N_des| <= tol_N.

The neighbour search itself (which particles have r_ij < h) is a library step here (scipy cKDTree with a periodic
box); everything else is written out.  Pins: tests/test_oracle_sph.py.  Only tests/ may import this module.
"""
from __future__ import annotations

import numpy as np
from scipy.spatial import cKDTree


def w_kernel(u):
    """R43: dimensionless cubic spline, support u <= 1."""
    u = np.asarray(u, np.float64)
    return np.where(u <= 0.5, 1.0 - 6.0 * u * u + 6.0 * u * u * u, np.where(u <= 1.0, 2.0 * (1.0 - u) ** 3, 0.0))


def neighbour_number(r, h):
    """R44 for one target: r = distances to all candidates (self included as r = 0)."""
    return (4.0 * np.pi / 3.0) * (8.0 / np.pi) * float(w_kernel(np.asarray(r) / h).sum())


def density_at(r, m, h):
    """R46 for one target."""
    return (8.0 / (np.pi * h ** 3)) * float((np.asarray(m) * w_kernel(np.asarray(r) / h)).sum())


def sph_density(pos, mass, L, n_des, targets=None, h_cap=None):
    """-> (h f64[n_t], rho f64[n_t], N f64[n_t]) for pos[targets] (all particles if None)."""
    pos = np.asarray(pos, np.float64)
    mass = np.asarray(mass, np.float64)
    n = pos.shape[0]
    L = float(L)
    tidx = np.arange(n) if targets is None else np.asarray(targets, np.int64)
    tree = cKDTree(np.mod(pos, L), boxsize=L)
    # candidates: everything within a radius that certainly holds the root (N(h) >= number of particles within h / 2,
    # since w(u) >= 1/4 for u <= 1/2 and (4 pi / 3)(8 / pi) / 4 = 8/3 > 1: the ball of the 2^k-th ... grown until N >= n_des)
    h_out = np.empty(tidx.shape[0])
    rho = np.empty(tidx.shape[0])
    nn = np.empty(tidx.shape[0])
    h0 = (3.0 * n_des * L ** 3 / (4.0 * np.pi * n)) ** (1.0 / 3.0)
    cap = 0.5 * L * (1 - 1e-12) if h_cap is None else float(h_cap)
    for k, i in enumerate(tidx):
        hi = min(h0, cap)
        while True:
            idx = tree.query_ball_point(np.mod(pos[i], L), hi)
            d = pos[idx] - pos[i]
            d -= L * np.round(d / L)
            r = np.sqrt((d * d).sum(1))
            if neighbour_number(r, hi) >= n_des or hi >= cap:
                break
            hi = min(2.0 * hi, cap)
        m = mass[idx]
        lo = 0.0
        for _ in range(200):                       # bisection on the candidates within hi (a superset for any h <= hi)
            mid = 0.5 * (lo + hi)
            if neighbour_number(r, mid) < n_des:
                lo = mid
            else:
                hi = mid
            if hi - lo <= 1e-14 * hi:
                break
        h = 0.5 * (lo + hi)
        h_out[k] = h
        rho[k] = density_at(r, m, h)
        nn[k] = neighbour_number(r, h)
    return h_out, rho, nn
