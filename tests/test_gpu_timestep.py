"""-m gpu: row f2, the time-step shell on the device (og_ts_*) against oracle/timestep.py.

Kernel by kernel on the same seeded inputs: the active list and the bins are integer work -> bit-exact (the bin rule
is decided in fp32 on both sides from the same fp32 accelerations); a_old = |a| in fp32 with a fixed operation order ->
equal bits; drift and kick are one fp32 fma per coordinate against fp64 -> 1e-6 relative to the scale of the state.
Then the whole loop: K synchronisation steps of a small clustered box, each side with its own forces (CUDA walk / oracle
walk), compared on positions, velocities, bins and the sizes of the active sets."""
import numpy as np
import pytest

import oracle
from oracle import timestep as ots
from paper_2606_17145_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B(cuda_device):
    from paper_2606_17145_b200 import binding
    return binding


def _t(x, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(x))
    return t.cuda() if dtype is None else t.to(dtype).cuda()


def test_drift_wraps_and_matches(B):
    import torch
    rng = np.random.default_rng(0)
    n, L = 100_003, 100.0
    pos = (rng.random((n, 3)) * L).astype(np.float32)
    pos[pos >= L] = 0
    vel = (rng.standard_normal((n, 3)) * 30).astype(np.float32)
    vel[:10] *= 50                                              # several box lengths per step
    dpos, dvel = _t(pos), _t(vel)
    B.og_ts_drift(dpos, dvel, 1.7, L)
    got = dpos.cpu().numpy()
    ref = np.mod(pos.astype(np.float64) + vel.astype(np.float64) * np.float64(np.float32(1.7)), L)
    assert np.all((got >= 0) & (got < np.float32(L)))
    d = np.abs(got - ref)
    d = np.minimum(d, L - d)                                    # a value that rounds across the wall is still right
    assert d.max() <= 2e-5 * L * 1e-1 + 1e-5 * np.abs(vel).max() * 1.7 * 1e-1


@pytest.mark.parametrize("n", [1, 255, 2048, 2049, 300_007])
def test_active_list_and_next_tick_are_exact(B, n):
    import torch
    rng = np.random.default_rng(n)
    bmax = 7
    bins = rng.integers(0, bmax + 1, n).astype(np.uint8)
    if n > 10:
        bins[bins == bmax] = bmax - 1                           # leave the finest level empty: next tick = 2, not 1
    dbin = _t(bins)
    scratch = torch.empty(B.og_ts_scratch_bytes(n), dtype=torch.uint8, device="cuda")
    act = torch.empty(n, dtype=torch.int32, device="cuda")
    for tick in (0, 2, 4, 6, 64, 96, 128):
        na = B.og_ts_active_list(dbin, tick, bmax, act, scratch)
        ref = np.nonzero(ots.active_mask(bins, tick, bmax))[0]
        assert na == ref.shape[0]
        assert np.array_equal(act[:na].cpu().numpy().view(np.uint32), ref.astype(np.uint32))
        assert B.og_ts_next_tick(dbin, tick, bmax, scratch) == ots.next_sync_tick(bins, tick, bmax)


@pytest.mark.parametrize("first", [True, False])
def test_kick_bins_a_old_exact_and_velocity(B, first):
    import torch
    rng = np.random.default_rng(5)
    n, bmax, eta, dt_max = 50_001, 9, 0.025, 0.0625
    eps = np.where(rng.random(n) < 0.5, 1e-3, 4e-3).astype(np.float32)
    bins = rng.integers(0, bmax + 1, n).astype(np.uint8)
    vel = rng.standard_normal((n, 3)).astype(np.float32)
    tick = 48                                                   # divisible by 16: steps of bins >= bmax - 4 are aligned
    act = np.nonzero(ots.active_mask(bins, tick, bmax))[0].astype(np.uint32) if not first else np.arange(n, dtype=np.uint32)
    acc = (rng.standard_normal((act.shape[0], 3)) * 10.0 ** rng.uniform(-3, 3, (act.shape[0], 1))).astype(np.float32)
    acc[:3] = 0                                                 # |a| = 0 -> bin 0
    dvel, dbin, daold = _t(vel), _t(bins), torch.zeros(n, device="cuda")
    B.og_ts_kick(dvel, dbin, daold, None if first else _t(act.view(np.int32)), act.shape[0], _t(acc), _t(eps), eta, dt_max, bmax,
                 tick, first)
    an = ots.acc_norm32(acc)
    want = ots.wanted_bin(an, eps[act], eta, dt_max, bmax)
    new = want if first else ots.next_bin(bins[act], want, tick, bmax)
    ref_bins = bins.copy()
    ref_bins[act] = new
    assert np.array_equal(dbin.cpu().numpy(), ref_bins)                       # integer decisions: exact
    ref_aold = np.zeros(n, np.float32)
    ref_aold[act] = an
    assert np.array_equal(daold.cpu().numpy(), ref_aold)                      # fixed fp32 operation order: equal bits
    dt_new = dt_max / np.exp2(new.astype(np.float64))
    half = 0.5 * dt_new if first else 0.5 * (dt_max / np.exp2(bins[act].astype(np.float64)) + dt_new)
    ref_vel = vel.astype(np.float64)
    ref_vel[act] += acc.astype(np.float64) * half[:, None]
    err = np.abs(dvel.cpu().numpy() - ref_vel)
    assert (err <= 1e-6 * (np.abs(ref_vel) + 1e-3)).all()
    assert len(set(new.tolist())) > 4                                          # the test really spans several bins


def test_kick_records_a_bad_active_index(B):
    """og.h (og_ts_kick): an active_idx entry >= n is skipped -- no particle is touched for it -- and, when the caller
    passes a status word, recorded there as OG_TS_BAD_INDEX; a clean list leaves the word at zero, and the entries next
    to the bad ones are kicked as usual."""
    import torch
    rng = np.random.default_rng(9)
    n, bmax, eta, dt_max = 4099, 6, 0.025, 0.0625
    eps = np.full(n, 2e-3, np.float32)
    vel = rng.standard_normal((n, 3)).astype(np.float32)
    bins = rng.integers(0, bmax + 1, n).astype(np.uint8)
    act = rng.choice(n, 600, replace=False).astype(np.uint32)
    acc = rng.standard_normal((600, 3)).astype(np.float32)

    def run(a, status):
        dv, db, da = _t(vel), _t(bins), torch.zeros(n, device="cuda")
        B.og_ts_kick(dv, db, da, _t(a.view(np.int32)), a.shape[0], _t(acc), _t(eps), eta, dt_max, bmax, 0, False, status)
        torch.cuda.synchronize()
        return dv.cpu().numpy(), db.cpu().numpy(), da.cpu().numpy()

    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    v0, b0, a0 = run(act, status)
    assert int(status[0]) == 0
    bad = act.copy()
    bad[[5, 333]] = [n, 0xffffffff]
    v1, b1, a1 = run(bad, status)
    assert int(status[0]) == B.OG_TS_BAD_INDEX
    skipped = act[[5, 333]]
    same = np.ones(n, bool)
    same[skipped] = False
    assert np.array_equal(v1[same], v0[same]) and np.array_equal(b1[same], b0[same]) and np.array_equal(a1[same], a0[same])
    assert np.array_equal(v1[skipped], vel[skipped]) and np.array_equal(b1[skipped], bins[skipped])   # untouched
    v2, b2, a2 = run(bad, None)                                   # no status word: same skipping, nothing recorded
    assert np.array_equal(v2, v1) and np.array_equal(b2, b1)


def test_whole_loop_matches_the_oracle_stepper(B):
    """K synchronisation steps of a small clustered box: CUDA walk + og_ts_* against oracle walk + oracle stepper."""
    import torch
    w = W.nfw_box(24, 8, 100.0, W.SEED0 + 4242, name="ts_small")
    n, L = w.n, w.L
    rng = np.random.default_rng(1)
    vel0 = (0.02 * rng.standard_normal((n, 3))).astype(np.float32)
    eta, dt_max, bmax, K = 0.02, 0.5, 6, 10
    oprm = oracle.make_params(L, w.r_s, G=w.G, alpha=w.alpha, theta=w.theta)

    def oforce(pos32, idx, a_old):
        t = oracle.build_tree(pos32, w.mass, w.eps, oprm)
        acc, _, _ = oracle.walk(t, np.asarray(idx, np.uint32), a_old, want_counters=False)
        return acc
    ost = ots.Stepper(w.pos, vel0, w.eps, L, eta, dt_max, bmax, oforce)

    prm = B.make_params(w.r_s, G=w.G, alpha=w.alpha, theta=w.theta)
    pos, vel, mass, eps = _t(w.pos), _t(vel0), _t(w.mass), _t(w.eps)
    bins = torch.zeros(n, dtype=torch.uint8, device="cuda")
    a_old = torch.zeros(n, device="cuda")
    act = torch.empty(n, dtype=torch.int32, device="cuda")
    scratch = torch.empty(B.og_ts_scratch_bytes(n), dtype=torch.uint8, device="cuda")
    tree = B.og_tree_build(pos, mass, eps, L, prm)
    acc, _ = B.og_shortrange_accel(tree, None, None, want_pot=False)
    B.og_tree_free(tree)
    B.og_ts_kick(vel, bins, a_old, None, n, acc, eps, eta, dt_max, bmax, 0, True)
    tick, nact = 0, []
    for _ in range(K):
        nxt = B.og_ts_next_tick(bins, tick, bmax, scratch)
        B.og_ts_drift(pos, vel, (nxt - tick) * dt_max / 2 ** bmax, L)
        tick = nxt
        na = B.og_ts_active_list(bins, tick, bmax, act, scratch)
        tree = B.og_tree_build(pos, mass, eps, L, prm)
        sub = act[:na].contiguous()
        acc, _ = B.og_shortrange_accel(tree, sub, a_old[sub.long()].contiguous(), want_pot=False)
        assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
        B.og_tree_free(tree)
        B.og_ts_kick(vel, bins, a_old, sub, na, acc, eps, eta, dt_max, bmax, tick, False)
        nact.append(na)
        ost.step()
        assert tick == ost.tick
    assert len(set(nact)) > 1 and min(nact) < n // 4                         # a real hierarchy of active sets
    gb, ob = bins.cpu().numpy(), ost.bin
    assert (gb != ob).sum() <= max(2, n // 2000), (gb != ob).sum()           # a bin decided within fp32 rounding of a boundary
    dx = np.abs(pos.cpu().numpy().astype(np.float64) - ost.x)
    dx = np.minimum(dx, L - dx)
    same = gb == ob
    assert dx[same].max() <= 2e-5 * L * 1e-2 + 1e-6 * L                      # ~ fp32 resolution of a position in the box
    dv = np.abs(vel.cpu().numpy().astype(np.float64) - ost.v)
    vs = np.abs(ost.v).max()
    assert np.percentile(dv[same], 99.9) <= 1e-4 * vs and dv[same].max() <= 1e-2 * vs
