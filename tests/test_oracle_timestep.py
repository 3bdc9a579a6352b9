"""Pins for oracle/timestep.py (row f2: the time-step shell).  CPU only.  The references are
closed forms and exact properties of the leapfrog, not a second copy of the stepper."""
import math

import numpy as np
import pytest

import oracle
from oracle import timestep as ts


def _newton_force(L, mass, eps, rs_frac=1.0 / 9.1):
    """Short-range O(N^2) oracle in its Newtonian limit (r_s = L / 9.1, P5): pair force G m T(w) / r^2 with potential
    -G m erfc(w) / r, mutually consistent (P13)."""
    prm = oracle.make_params(L, L * rs_frac)

    def force(pos32, idx, a_old):
        acc, pot = oracle.direct(pos32, mass, eps, prm, np.asarray(idx, np.uint32))
        force.last_pot = pot
        return acc
    force.prm = prm
    return force


def _two_body(L=1.0, sep=0.01, m=1e-6):
    """Equal masses on a circular orbit around the box centre under the short-range pair force."""
    rs = L / 9.1
    w = sep / (2 * rs)
    T = math.erfc(w) + 2 * w / math.sqrt(math.pi) * math.exp(-w * w)
    a = m * T / sep ** 2                      # acceleration of each body towards the other
    v = math.sqrt(a * sep / 2)                # circular: v^2 / (sep / 2) = a
    pos = np.array([[0.5 - sep / 2, 0.5, 0.5], [0.5 + sep / 2, 0.5, 0.5]])
    vel = np.array([[0.0, -v, 0.0], [0.0, v, 0.0]])
    period = 2 * math.pi * (sep / 2) / v
    return pos, vel, np.full(2, m, np.float32), np.full(2, 1e-7, np.float32), period


def _energy(st, mass, force):
    idx = np.arange(st.x.shape[0], dtype=np.uint32)
    acc = force(st.pos32(), idx, None)
    v = st.synchronised_velocity(acc.astype(np.float32))
    m = mass.astype(np.float64)
    return 0.5 * (m * (v * v).sum(1)).sum() + 0.5 * (m * force.last_pot).sum()


def test_wanted_bin_closed_form_and_clamps():
    eta, dt_max, bmax = 0.025, 0.5, 10
    eps = np.full(8, 1e-3, np.float32)
    # |a| = 2 eta eps 4^k / dt_max^2 exactly representable for these values? use powers of two throughout
    eta, dt_max = 0.03125, 0.5
    base = np.float32(2 * eta * 1e-3 / dt_max ** 2)
    a = np.array([0.0, base, base * 1.0001, base * 4, base * 4.0001, base * 4 ** 5, base * 4 ** 9.5, base * 4 ** 20], np.float32)
    b = ts.wanted_bin(a, eps, eta, dt_max, bmax)
    assert list(b) == [0, 0, 1, 1, 2, 5, 10, 10]
    assert ts.wanted_bin(np.array([np.nan], np.float32), eps[:1], eta, dt_max, bmax)[0] == 0


def test_active_ticks_alignment_and_single_doubling():
    bmax = 4
    bins = np.array([0, 1, 2, 3, 4], np.uint8)
    seen = np.zeros(5, int)
    for tick in range(1, 17):
        seen += ts.active_mask(bins, tick, bmax)
    assert list(seen) == [1, 2, 4, 8, 16]                       # 2^b activations per dt_max
    assert ts.next_sync_tick(bins, 0, bmax) == 1 and ts.next_sync_tick(bins[:3], 4, bmax) == 8
    # grow: only by one level and only at a tick the larger step divides; shrink: freely
    cur = np.array([3, 3, 3, 1], np.uint8)
    want = np.array([0, 0, 4, 3], np.uint8)
    assert list(ts.next_bin(cur, want, 2, bmax)) == [3, 3, 4, 3]      # step of bin 2 = 4 ticks does not divide 2
    assert list(ts.next_bin(cur, want, 4, bmax)) == [2, 2, 4, 3]      # divides 4: one level up, not three


def test_free_particles_drift_all_and_wrap():
    L = 1.0
    pos = np.array([[0.1, 0.2, 0.95], [0.5, 0.5, 0.5]])
    vel = np.array([[0.3, -0.7, 0.4], [0.0, 0.0, 0.0]])
    st = ts.Stepper(pos, vel, np.full(2, 1e-3, np.float32), L, 0.025, 0.25, 3, lambda p, i, a: np.zeros((len(i), 3)))
    assert list(st.bin) == [0, 0]
    for _ in range(4):
        st.step()
    assert st.tick == 4 * 2 ** 3
    assert np.allclose(st.x, np.mod(pos + vel * 1.0, L), atol=1e-14) and np.all((st.x >= 0) & (st.x < L))


@pytest.mark.parametrize("adaptive", [False, True])
def test_circular_orbit_phase_error_is_second_order(adaptive):
    """Kick-drift-kick is second order: after one period of a circular two-body orbit the bodies are back at their
    start up to an O(dt^2) error (phase drift plus the epicycle of a start that is circular only for the exact flow),
    which quarters when dt halves (dt = P/16, P/32, P/64: far above the fp32 rounding of the positions handed to the
    force routine).  `adaptive`: the same steps as bin 2 of a
    5-level hierarchy (dt_max = 4 dt), which must give the same orbit."""
    errs = []
    for nstep in (16, 32, 64):
        pos, vel, mass, eps, period = _two_body()
        force = _newton_force(1.0, mass, eps)
        dt = period / nstep
        a = float(np.linalg.norm(force(pos.astype(np.float32), np.arange(2, dtype=np.uint32), None)[0]))
        if adaptive:
            dt_max, bmax = 4 * dt, 4
            eta = dt ** 2 * a / (2 * 1e-7) * 1.1            # the criterion allows a little more than dt: bin 2
        else:
            dt_max, bmax, eta = dt, 0, 1e30
        st = ts.Stepper(pos, vel, eps, 1.0, eta, dt_max, bmax, force)
        assert list(st.bin) == ([2, 2] if adaptive else [0, 0])
        for _ in range(nstep):
            st.step()
        assert st.tick == nstep * (4 if adaptive else 1) and list(st.kicks) == [nstep, nstep]
        errs.append(float(np.abs(st.x - pos).max() / 0.005))
    print(errs)
    assert errs[0] < 0.5 and 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5, errs


def test_time_reversibility_with_fixed_steps():
    rng = np.random.default_rng(3)
    n, L = 24, 1.0
    pos = 0.5 + 0.02 * rng.standard_normal((n, 3))
    vel = 1e-3 * rng.standard_normal((n, 3))
    mass = np.full(n, 1e-6, np.float32)
    eps = np.full(n, 2e-3, np.float32)
    force = _newton_force(L, mass, eps)
    st = ts.Stepper(pos, vel, eps, L, 1e30, 0.05, 0, force)          # one bin: fixed steps
    for _ in range(20):
        st.step()
    idx = np.arange(n, dtype=np.uint32)
    acc = force(st.pos32(), idx, None).astype(np.float32)
    v_sync = st.synchronised_velocity(acc)
    back = ts.Stepper(st.x, -v_sync, eps, L, 1e30, 0.05, 0, force)
    for _ in range(20):
        back.step()
    # positions are handed to the force routine in fp32, so reversibility holds to fp32 rounding of the forces
    assert np.abs(back.x - pos).max() < 1e-7


def test_hierarchical_bins_kick_counts_and_a_old():
    """A tight pair (large |a|, small step) and two distant free-floaters (bin 0): over one dt_max the pair is kicked
    2^b times, the others once; a_old holds the fp32 |a| of the last evaluation."""
    pos, vel, mass, eps, period = _two_body()
    pos = np.vstack([pos, [[0.1, 0.1, 0.1], [0.9, 0.9, 0.1]]])
    vel = np.vstack([vel, np.zeros((2, 3))])
    mass = np.full(4, 1e-6, np.float32)
    eps = np.full(4, 1e-7, np.float32)
    force = _newton_force(1.0, mass, eps)
    a_pair = float(np.linalg.norm(force(pos[:2].astype(np.float32), np.arange(2, dtype=np.uint32), None)[0]))
    force = _newton_force(1.0, mass, eps)
    dt_max = period / 8
    eta = (dt_max / 8) ** 2 * a_pair / (2 * 1e-7) * 1.1                # the pair may take a little more than dt_max / 8: bin 3
    st = ts.Stepper(pos, vel, eps, 1.0, eta, dt_max, 5, force)
    assert list(st.bin[:2]) == [3, 3] and list(st.bin[2:]) == [0, 0]
    nact = []
    while st.tick < 2 ** 5:
        act = st.step()
        nact.append(len(act))
    assert list(st.kicks) == [8, 8, 1, 1]
    assert nact == [2] * 7 + [4]
    acc = force(st.pos32(), np.arange(4, dtype=np.uint32), None)
    assert np.allclose(st.a_old, ts.acc_norm32(acc.astype(np.float32)), rtol=1e-6)
