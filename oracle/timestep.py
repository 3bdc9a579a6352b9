"""oracle.timestep -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain NumPy restatement of the time-step shell around the force calls (PAPER.md:80 time bins
with few active particles, :82 "we execute the particle drifting process at the onset of a GPU-ported timestep for all
particles (i.e., active and non-active ones)", :320 find_sync_point_and_drift).  The paper prints no formula; the rules
are Gadget-2's individual power-of-two time steps (Springel 2005, the paper's citation P:296) -- readings R37..R42 of
DESIGN.md Sec. 11:

  R37  integer timeline: one tick = dt_max / 2^bmax; a particle in bin b has a step of 2^(bmax - b) ticks
       (dt_b = dt_max / 2^b) and is ACTIVE at the ticks its step divides; the system advances to the next tick at which
       some particle is active.
  R38  wanted bin from dt_i = sqrt(2 eta eps_i / |a_i|): the smallest b in [0, bmax] with 4^b >= dt_max^2 |a| / (2 eta eps),
       decided in fp32 in the stated operation order (a floating-point value decides an integer: both sides take the
       decision in the same precision); a step may always shrink, and may grow by ONE level only at a tick the larger
       step divides.
  R39  drift: every particle (active or not) is moved to the new time, x += v dt, wrapped into [0, L).
  R40  kick-drift-kick: an active particle gets the closing half kick of its old step and the opening half kick of its
       new step, v += a (dt_old + dt_new) / 2, with the acceleration just computed at the drifted positions.
  R41  a_old of a particle = |a| of its last force evaluation (fp32), the input of the relative opening criterion.
  R42  the tree is rebuilt from the drifted positions at every step (the reference drifts its CPU-built nodes instead,
       P:320 force_drift_node; on the device a rebuild costs less than a tenth of a full walk).

State arithmetic is fp64 here (positions are rounded to fp32 when handed to a force routine, whose inputs are fp32).
Pins: tests/test_oracle_timestep.py.  Only tests/ may import this module; it shares no code with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def acc_norm32(acc) -> np.ndarray:
    """|a| in fp32, operation order fixed: ((ax*ax + ay*ay) + az*az), one rounding per operation, IEEE sqrt."""
    a = np.asarray(acc, np.float32)
    s = (a[:, 0] * a[:, 0] + a[:, 1] * a[:, 1]).astype(np.float32)
    s = (s + a[:, 2] * a[:, 2]).astype(np.float32)
    return np.sqrt(s, dtype=np.float32)


def wanted_bin(anorm32, eps32, eta, dt_max, bmax) -> np.ndarray:
    """R38, fp32: ratio = ((dt_max * dt_max) * |a|) / ((2 * eta) * eps); b = smallest integer in [0, bmax] with 4^b >= ratio."""
    f = np.float32
    num = (f(f(dt_max) * f(dt_max)) * np.asarray(anorm32, f)).astype(f)
    den = (f(f(2.0) * f(eta)) * np.asarray(eps32, f)).astype(f)
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = (num / den).astype(f)
    b = np.zeros(ratio.shape, np.int64)
    p = f(1.0)
    for k in range(int(bmax)):
        b += (ratio > p)            # 4^k < ratio -> at least k + 1   (NaN compares false: bin 0)
        p = f(p * f(4.0))
    return b.astype(np.uint8)


def step_ticks(b, bmax):
    return np.left_shift(np.int64(1), (int(bmax) - np.asarray(b, np.int64)))


def active_mask(bins, tick, bmax) -> np.ndarray:
    """R37: particle i is active at `tick` iff its step divides it."""
    return (np.int64(tick) % step_ticks(bins, bmax)) == 0


def next_bin(cur, want, tick, bmax) -> np.ndarray:
    """R38: shrink freely; grow by one level only if the larger step divides `tick`."""
    cur = np.asarray(cur, np.int64)
    want = np.asarray(want, np.int64)
    nb = np.where(want >= cur, want, cur)                       # smaller or equal step: take the wanted bin
    grow = (want < cur) & ((np.int64(tick) % step_ticks(np.maximum(cur - 1, 0), bmax)) == 0)
    nb = np.where(grow, cur - 1, nb)
    return nb.astype(np.uint8)


def next_sync_tick(bins, tick, bmax) -> int:
    """R37: the next tick (> tick) at which some particle is active."""
    s = step_ticks(bins, bmax)
    return int((np.int64(tick) // s + 1).__mul__(s).min())


class Stepper:
    """Kick-drift-kick with individual time steps and drift-all.  force(pos32, active_idx, a_old32_active | None)
    -> acc[n_active][3]; it is called with None at the start (no a_old yet: geometric criterion)."""

    def __init__(self, pos, vel, eps, L, eta, dt_max, bmax, force):
        self.x = np.asarray(pos, np.float64).copy()
        self.v = np.asarray(vel, np.float64).copy()
        self.eps = np.asarray(eps, np.float32)
        self.L, self.eta, self.dt_max, self.bmax, self.force = float(L), float(eta), float(dt_max), int(bmax), force
        n = self.x.shape[0]
        self.tick = 0
        self.tick_dt = self.dt_max / 2 ** self.bmax
        self.kicks = np.zeros(n, np.int64)
        idx = np.arange(n, dtype=np.uint32)
        acc = np.asarray(self.force(self.pos32(), idx, None), np.float64)
        acc32 = acc.astype(np.float32)
        self.a_old = acc_norm32(acc32)
        self.bin = wanted_bin(self.a_old, self.eps, self.eta, self.dt_max, self.bmax)
        self.v += acc32.astype(np.float64) * (0.5 * self.dt_of(self.bin))[:, None]          # opening half kick
        self.n_active_last = n

    def pos32(self):
        p = self.x.astype(np.float32)
        p[p >= np.float32(self.L)] = 0.0
        return p

    def dt_of(self, b):
        return self.dt_max / np.exp2(np.asarray(b, np.float64))

    def step(self):
        t1 = next_sync_tick(self.bin, self.tick, self.bmax)
        dt = (t1 - self.tick) * self.tick_dt
        self.x = np.mod(self.x + self.v * dt, self.L)                                       # R39: drift all
        self.tick = t1
        act = np.nonzero(active_mask(self.bin, t1, self.bmax))[0].astype(np.uint32)
        acc32 = np.asarray(self.force(self.pos32(), act, self.a_old[act]), np.float64).astype(np.float32)
        an = acc_norm32(acc32)
        old = self.bin[act]
        new = next_bin(old, wanted_bin(an, self.eps[act], self.eta, self.dt_max, self.bmax), t1, self.bmax)
        self.v[act] += acc32.astype(np.float64) * (0.5 * (self.dt_of(old) + self.dt_of(new)))[:, None]   # R40
        self.bin[act] = new
        self.a_old[act] = an                                                                # R41
        self.kicks[act] += 1
        self.n_active_last = int(act.shape[0])
        return act

    def synchronised_velocity(self, acc_all):
        """Velocities at the current time for diagnostics: remove the opening half kick (needs a at the current
        positions for every particle)."""
        return self.v - np.asarray(acc_all, np.float64) * (0.5 * self.dt_of(self.bin))[:, None]
