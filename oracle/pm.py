"""oracle.pm -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain fp64 NumPy restatement of the particle-mesh LONG-RANGE part of the TreePM force (
PAPER.md:124: "the long-range gravitational forces from the PM, which uses FFTW ... runs on CPU only").  The paper
prints no formula; the steps are the Gadget-2 PM scheme (Springel 2005, the paper's citation P:296) with the force
split at r_s that the short-range walk uses (readings R31..R36), written out step by step:

  R31  CIC assignment of the particle masses to the Ng^3 grid points x_g = g L / Ng (periodic).
  R32  phi_k = -4 pi G / (V k^2) * exp(-k^2 r_s^2) * M_k / W(k)^2,  M_k = DFT of the mass grid, V = L^3,
       k = 2 pi n / L with n in (-Ng/2, Ng/2]^3, phi_0 = 0;  W(k) = prod_i sinc^2(k_i Delta / 2) is the CIC window,
       divided out twice (assignment and interpolation).
  R33  phi on the grid by the inverse DFT; acceleration on the grid by the 4-point finite difference
       a = -[ (4/3) (phi_{+1} - phi_{-1}) / (2 Delta) - (1/3) (phi_{+2} - phi_{-2}) / (4 Delta) ] per axis.
  R34  CIC interpolation of a and phi from the 8 surrounding grid points to the particle.

A library primitive (numpy.fft) serves as the DFT step.  Pins (tests/test_oracle_pm.py): the exact long-range
k-space sum by brute force (PM converges to it as r_s / Delta grows), short + long = Ewald, sum m a = 0, zero force
on a lattice commensurate with the grid, zero self-force.

Only tests/ and bench-side measurement may import this module; it shares no code with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def cic_deposit(pos, mass, L, ng):
    """R31: mass grid M[g] (fp64), grid points at g L / ng."""
    x = np.asarray(pos, np.float64) * (ng / float(L))
    i0 = np.floor(x).astype(np.int64)
    f = x - i0
    grid = np.zeros((ng, ng, ng), np.float64)
    m = np.asarray(mass, np.float64)
    for dx in (0, 1):
        wx = f[:, 0] if dx else 1.0 - f[:, 0]
        ix = (i0[:, 0] + dx) % ng
        for dy in (0, 1):
            wy = f[:, 1] if dy else 1.0 - f[:, 1]
            iy = (i0[:, 1] + dy) % ng
            for dz in (0, 1):
                wz = f[:, 2] if dz else 1.0 - f[:, 2]
                iz = (i0[:, 2] + dz) % ng
                np.add.at(grid, (ix, iy, iz), m * wx * wy * wz)
    return grid


def potential_grid(mgrid, L, r_s, G=1.0):
    """R32, R33 (first half): long-range potential on the grid points."""
    ng = mgrid.shape[0]
    L = float(L)
    delta = L / ng
    n1 = np.fft.fftfreq(ng, d=1.0 / ng)              # integers in (-ng/2, ng/2]  (the Nyquist row carries -ng/2)
    nz = np.fft.rfftfreq(ng, d=1.0 / ng)
    kx = (2.0 * np.pi / L) * n1[:, None, None]
    ky = (2.0 * np.pi / L) * n1[None, :, None]
    kz = (2.0 * np.pi / L) * nz[None, None, :]
    k2 = kx * kx + ky * ky + kz * kz
    # np.sinc(x) = sin(pi x) / (pi x):  sinc(k Delta / 2) = np.sinc(k Delta / (2 pi)) = np.sinc(n / ng)
    w = (np.sinc(n1[:, None, None] / ng) * np.sinc(n1[None, :, None] / ng) * np.sinc(nz[None, None, :] / ng)) ** 2
    mk = np.fft.rfftn(mgrid)
    with np.errstate(divide="ignore", invalid="ignore"):
        green = -4.0 * np.pi * G / (L ** 3 * k2) * np.exp(-k2 * r_s * r_s) / (w * w)
    green[0, 0, 0] = 0.0
    # sum_k phi_k exp(i k x_g) = ng^3 * irfftn(phi_k)
    return np.fft.irfftn(green * mk, s=mgrid.shape, axes=(0, 1, 2)) * ng ** 3, delta


def accel_grids(phi, delta):
    """R33 (second half): 4-point finite difference, a = -grad phi."""
    out = []
    for ax in range(3):
        d1 = np.roll(phi, -1, ax) - np.roll(phi, 1, ax)
        d2 = np.roll(phi, -2, ax) - np.roll(phi, 2, ax)
        out.append(-((4.0 / 3.0) * d1 / (2.0 * delta) - (1.0 / 3.0) * d2 / (4.0 * delta)))
    return out


def cic_interp(grid, pos, L):
    """R34: value of a grid field at the particle positions."""
    ng = grid.shape[0]
    x = np.asarray(pos, np.float64) * (ng / float(L))
    i0 = np.floor(x).astype(np.int64)
    f = x - i0
    out = np.zeros(x.shape[0], np.float64)
    for dx in (0, 1):
        wx = f[:, 0] if dx else 1.0 - f[:, 0]
        ix = (i0[:, 0] + dx) % ng
        for dy in (0, 1):
            wy = f[:, 1] if dy else 1.0 - f[:, 1]
            iy = (i0[:, 1] + dy) % ng
            for dz in (0, 1):
                wz = f[:, 2] if dz else 1.0 - f[:, 2]
                iz = (i0[:, 2] + dz) % ng
                out += wx * wy * wz * grid[ix, iy, iz]
    return out


def pm_longrange(pos, mass, L, r_s, ng, G=1.0, targets=None):
    """Long-range acceleration and potential at the particles (or at pos[targets]).
    -> acc f64[n_t][3], pot f64[n_t]"""
    pos = np.asarray(pos, np.float64)
    mgrid = cic_deposit(pos, mass, L, ng)
    phi, delta = potential_grid(mgrid, L, r_s, G)
    tp = pos if targets is None else pos[np.asarray(targets)]
    acc = np.stack([cic_interp(a, tp, L) for a in accel_grids(phi, delta)], axis=1)
    return acc, cic_interp(phi, tp, L)
