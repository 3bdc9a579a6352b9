"""Seeded synthetic inputs (BASELINE.json `configs`, readings of SURVEY.md Sec. 8.4).

This module holds NONE of the method's arithmetic: it only draws particle
positions, masses, softenings and active subsets.  It is the one module that both
the oracle's tests and the CUDA path's tests / bench use, so that both sides see
bit-identical fp32 arrays (R4: positions are generated in fp64, rounded once to
fp32, and that fp32 array is the input of both sides).

The paper's own workloads -- Magneticum Box1a/mr, the Dianoga zoom
(PAPER.md:140-148), homogeneous 2x256^3..1024^3 ICs -- are not in the
container; these are their stand-ins (clustered box <-> `nfw256`, `nfw512`; early
homogeneous box <-> `lattice128`; two-species zoom with few active particles <->
`zoom`; tiny cross-check <-> `uniform32`).

Generator: numpy Generator(PCG64(seed)), seeds 260617145 + 1000 k for config k
(+1 for active subsets).
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

SEED0 = 260617145


@dataclass
class Workload:
    name: str
    pos: np.ndarray          # f32 [N][3], 0 <= x < L
    mass: np.ndarray         # f32 [N]
    eps: np.ndarray          # f32 [N]  Plummer-equivalent softening
    L: float
    r_s: float
    alpha: float = 0.005
    theta: float = 0.5
    rcut_over_rs: float = 4.5
    G: float = 1.0
    active_idx: np.ndarray | None = None   # u32, original indices; None -> all active

    @property
    def n(self) -> int:
        return int(self.pos.shape[0])

    @property
    def n_active(self) -> int:
        return self.n if self.active_idx is None else int(self.active_idx.shape[0])


def _finish(x64: np.ndarray, L: float) -> np.ndarray:
    """fp64 positions -> periodic wrap -> one rounding to fp32 -> x = 0 if x >= L."""
    x = np.mod(x64, L).astype(np.float32)
    x[x >= np.float32(L)] = np.float32(0.0)
    return np.ascontiguousarray(x)


def _nfw_m(x):
    return np.log1p(x) - x / (1.0 + x)


_NFW_X = np.linspace(0.0, 10.0, 1 << 16)
_NFW_M = _nfw_m(_NFW_X)


def _nfw_radii(rng, n, c):
    """n radii in units of the scale radius, inverse CDF of m(x) on [0, c]."""
    u = rng.random(n) * _nfw_m(c)
    return np.interp(u, _NFW_M, _NFW_X)


def _isotropic(rng, n):
    mu = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    st = np.sqrt(1.0 - mu * mu)
    return np.stack([st * np.cos(phi), st * np.sin(phi), mu], axis=1)


# --------------------------------------------------------------------------- #
def uniform_box(n_side: int = 32, L: float = 1.0, seed: int = SEED0 + 1000,
                name: str | None = None) -> Workload:
    """configs[0]: n_side^3 equal-mass particles, uniform random, eps = 0.02 L/n_side,
    r_s = 1.25 L/(2 n_side)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_side ** 3
    pos = _finish(rng.random((n, 3)) * L, L)
    mass = np.full(n, 1.0 / n, np.float32)
    eps = np.full(n, 0.02 * L / n_side, np.float32)
    return Workload(name or f"uniform{n_side}", pos, mass, eps, L, 1.25 * L / (2 * n_side))


def perturbed_lattice(n_side: int = 128, L: float = 1.0, seed: int = SEED0 + 2000,
                      rms_cells: float = 0.2, name: str | None = None) -> Workload:
    """configs[1]: lattice (i+1/2) L/n + Zel'dovich-style displacement from a Gaussian field
    with P(k) ~ k^-2, Nyquist planes zeroed, scaled to 3-D rms `rms_cells` grid spacings."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = n_side
    white = rng.standard_normal((n, n, n))
    dk = np.fft.rfftn(white)
    kx = np.fft.fftfreq(n, d=1.0 / n)
    kz = np.fft.rfftfreq(n, d=1.0 / n)
    KX, KY, KZ = np.meshgrid(kx, kx, kz, indexing="ij")
    k2 = KX * KX + KY * KY + KZ * KZ
    k2[0, 0, 0] = 1.0
    dk = dk / np.sqrt(k2)           # delta_k ~ k^-1  =>  P ~ k^-2
    dk[0, 0, 0] = 0.0
    nyq = n // 2
    dk[nyq, :, :] = 0.0
    dk[:, nyq, :] = 0.0
    dk[:, :, nyq] = 0.0
    psi = []
    for K in (KX, KY, KZ):
        psi.append(np.fft.irfftn(1j * K * dk / k2, s=(n, n, n), axes=(0, 1, 2)))
    psi = np.stack(psi, axis=-1).reshape(-1, 3)
    rms3 = np.sqrt(np.mean(np.sum(psi * psi, axis=1)))
    psi *= (rms_cells * L / n) / rms3
    g = (np.arange(n) + 0.5) * (L / n)
    GX, GY, GZ = np.meshgrid(g, g, g, indexing="ij")
    lat = np.stack([GX, GY, GZ], axis=-1).reshape(-1, 3)
    pos = _finish(lat + psi, L)
    N = n ** 3
    mass = np.full(N, 1.0 / N, np.float32)
    eps = np.full(N, 0.025 * L / n, np.float32)
    return Workload(name or f"lattice{n}", pos, mass, eps, L, 1.25 * L / n)


def nfw_box(n_side: int = 256, n_halos: int = 2000, L: float = 100.0,
            seed: int = SEED0 + 3000, halo_frac: float = 0.7, active_frac: float | None = None,
            name: str | None = None) -> Workload:
    """configs[2] / configs[4]: halo_frac of the mass in n_halos NFW halos (dN/dM ~ M^-1.9 on
    [1e-5, 1e-2] of the total, renormalised to halo_frac, c ~ U[5,10], truncated at r200,
    centres uniform), rest uniform.  eps = 0.02 L/n_side, r_s = 1.25 L/n_side."""
    rng = np.random.Generator(np.random.PCG64(seed))
    N = n_side ** 3
    g = 1.9
    a, b = 1e-5, 1e-2
    u = rng.random(n_halos)
    Mh = (a ** (1 - g) + u * (b ** (1 - g) - a ** (1 - g))) ** (1.0 / (1 - g))
    Mh *= halo_frac / Mh.sum()
    n_halo_part = int(round(halo_frac * N))
    raw = Mh / Mh.sum() * n_halo_part
    cnt = np.floor(raw).astype(np.int64)
    rem = n_halo_part - int(cnt.sum())
    order = np.argsort(-(raw - cnt), kind="stable")
    cnt[order[:rem]] += 1
    conc = rng.uniform(5.0, 10.0, n_halos)
    centre = rng.random((n_halos, 3)) * L
    pos = np.empty((N, 3), np.float32)
    o = 0
    for hidx in range(n_halos):
        m = int(cnt[hidx])
        if m == 0:
            continue
        f = m / N
        r200 = L * (3.0 * f / (800.0 * np.pi)) ** (1.0 / 3.0)
        r = _nfw_radii(rng, m, conc[hidx]) * (r200 / conc[hidx])
        x = centre[hidx][None, :] + r[:, None] * _isotropic(rng, m)
        pos[o:o + m] = _finish(x, L)
        o += m
    nb = N - o
    pos[o:] = _finish(rng.random((nb, 3)) * L, L)
    mass = np.full(N, 1.0 / N, np.float32)
    eps = np.full(N, 0.02 * L / n_side, np.float32)
    act = None
    if active_frac is not None:
        rng_a = np.random.Generator(np.random.PCG64(seed + 1))
        na = int(active_frac * N)
        act = np.sort(rng_a.choice(N, na, replace=False)).astype(np.uint32)
    return Workload(name or f"nfw{n_side}", pos, mass, eps, L, 1.25 * L / n_side, active_idx=act)


def zoom(n_hi: int = 8_388_608, n_lo: int = 2_097_152, L: float = 100.0,
         seed: int = SEED0 + 4000, active_frac: float = 0.05, rs_cells: int = 512,
         name: str | None = None) -> Workload:
    """configs[3]: two-species zoom.  hi-res (mass m): 40% in one NFW halo (c = 6, centred at the
    box centre, truncated at 0.1 L), 60% uniform in the sphere of radius 0.1 L; lo-res (mass 8m)
    uniform outside that sphere.  eps_hi = 0.001 L, eps_lo = 0.004 L, r_s = 1.25 L/rs_cells.
    Active: seeded random active_frac of the hi-res particles, sorted."""
    rng = np.random.Generator(np.random.PCG64(seed))
    R = 0.1 * L
    ctr = np.full(3, 0.5 * L)
    n_h = int(round(0.4 * n_hi))
    c = 6.0
    r = _nfw_radii(rng, n_h, c) * (R / c)
    x_h = ctr[None, :] + r[:, None] * _isotropic(rng, n_h)
    n_u = n_hi - n_h
    ru = R * rng.random(n_u) ** (1.0 / 3.0)
    x_u = ctr[None, :] + ru[:, None] * _isotropic(rng, n_u)
    lo = np.empty((n_lo, 3), np.float64)
    filled = 0
    while filled < n_lo:
        m = int((n_lo - filled) * 1.02) + 16
        cand = rng.random((m, 3)) * L
        keep = cand[np.sum((cand - ctr) ** 2, axis=1) > R * R]
        k = min(keep.shape[0], n_lo - filled)
        lo[filled:filled + k] = keep[:k]
        filled += k
    pos = _finish(np.concatenate([x_h, x_u, lo], axis=0), L)
    m_hi = 1.0 / (n_hi + 8 * n_lo)
    mass = np.concatenate([np.full(n_hi, m_hi), np.full(n_lo, 8 * m_hi)]).astype(np.float32)
    eps = np.concatenate([np.full(n_hi, 0.001 * L), np.full(n_lo, 0.004 * L)]).astype(np.float32)
    rng_a = np.random.Generator(np.random.PCG64(seed + 1))
    na = int(active_frac * n_hi)
    act = np.sort(rng_a.choice(n_hi, na, replace=False)).astype(np.uint32)
    return Workload(name or "zoom", pos, mass, eps, L, 1.25 * L / rs_cells, active_idx=act)


# --------------------------------------------------------------------------- #
# BASELINE.json configs, by name.  `small=True` gives the scaled-down variant the
# parity tests use (same recipe and structure, oracle finishes in seconds).
CONFIG_NAMES = ("uniform32", "lattice128", "nfw256", "zoom", "nfw512", "nfw512_active10")


def make(name: str, small: bool = False) -> Workload:
    if name == "uniform32":
        return uniform_box(16 if small else 32)
    if name == "lattice128":
        return perturbed_lattice(32 if small else 128)
    if name == "nfw256":
        return nfw_box(48, 40) if small else nfw_box(256, 2000, 100.0, SEED0 + 3000)
    if name == "zoom":
        if small:
            return zoom(1 << 17, 1 << 15, rs_cells=128, name="zoom_small")
        return zoom()
    if name == "nfw512":
        return nfw_box(64, 250, 400.0, SEED0 + 5000, name="nfw512_small") if small else \
            nfw_box(512, 16000, 400.0, SEED0 + 5000, name="nfw512")
    if name == "nfw512_active10":
        if small:
            return nfw_box(64, 250, 400.0, SEED0 + 5000, active_frac=0.1, name="nfw512a_small")
        return nfw_box(512, 16000, 400.0, SEED0 + 5000, active_frac=0.1, name="nfw512_active10")
    raise KeyError(name)
