"""-m gpu: row f1, the PM long-range force on the device (og_pm_*) against oracle/pm.py (fp64 NumPy restatement of
the same steps R31..R34) on the same seeded inputs, element by element; plus the physical check the row exists for:
short-range (og_shortrange_accel) + long-range (og_pm_longrange) against the exact periodic Newtonian force of
the oracle side (O(N^2) short-range sum + exact long-range k-space sum = Ewald, pinned in tests/test_oracle_pm.py).

Tolerance: the CUDA path is fp32 end to end (atomic mass assignment, cuFFT single precision,
finite differences of the potential), the oracle fp64; the error is measured against the rms long-range
acceleration: p99 <= 1e-4, max <= 1e-3 of a_rms; potential p99 <= 1e-4, max <= 1e-3 of max |phi|."""
import numpy as np
import pytest

import oracle
from oracle import pm as opm
from paper_2606_17145_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B(cuda_device):
    from paper_2606_17145_b200 import binding
    return binding


def _pm_gpu(B, w, ng, r_s, active=None):
    import torch
    pos, mass = torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.mass).cuda()
    pm = B.og_pm_create(ng, w.L, r_s, w.G)
    act = None if active is None else torch.from_numpy(np.asarray(active, np.uint32).view(np.int32)).cuda()
    a, p = B.og_pm_longrange(pm, pos, mass, act)
    a2, p2 = B.og_pm_longrange(pm, pos, mass, act)          # the handle is reusable
    torch.cuda.synchronize()
    B.og_pm_free(pm)
    return a.cpu().numpy().astype(np.float64), p.cpu().numpy().astype(np.float64), a2.cpu().numpy(), p2.cpu().numpy()


def _check(a, p, ao, po, what):
    arms = np.sqrt((ao ** 2).sum(1).mean())
    e = np.linalg.norm(a - ao, axis=1) / arms
    ep = np.abs(p - po) / np.abs(po).max()
    assert np.all(np.isfinite(a)) and np.all(np.isfinite(p))
    assert np.percentile(e, 99) <= 1e-4 and e.max() <= 1e-3, (what, np.percentile(e, 99), e.max())
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-3, (what, np.percentile(ep, 99), ep.max())
    return float(np.percentile(e, 99)), float(e.max())


@pytest.mark.parametrize("name,ng", [("uniform32", 32), ("nfw256", 64), ("lattice128", 32), ("zoom", 64)])
def test_pm_matches_oracle(B, name, ng):
    w = W.make(name, small=True)
    r_s = 1.25 * w.L / ng
    a, p, a2, p2 = _pm_gpu(B, w, ng, r_s)
    ao, po = opm.pm_longrange(w.pos, w.mass, w.L, float(np.float32(r_s)), ng, G=w.G)
    _check(a, p, ao, po, name)
    # a second call on the same handle agrees to fp32 rounding (atomic assignment order is free)
    arms = np.sqrt((ao ** 2).sum(1).mean())
    assert np.abs(a2 - a).max() <= 1e-4 * arms


def test_pm_active_subset_ragged_and_bad_index(B):
    import torch
    w = W.make("nfw256", small=True)
    ng, r_s = 32, 1.25 * w.L / 32
    rng = np.random.default_rng(5)
    act = rng.choice(w.n, 1001, replace=False).astype(np.uint32)        # unsorted, ragged
    a, p, _, _ = _pm_gpu(B, w, ng, r_s, act)
    ao, po = opm.pm_longrange(w.pos, w.mass, w.L, float(np.float32(r_s)), ng, G=w.G, targets=act)
    _check(a, p, ao, po, "subset")
    pm = B.og_pm_create(ng, w.L, r_s)
    pos, mass = torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.mass).cuda()
    empty = torch.empty(0, dtype=torch.int32, device="cuda")
    a0, p0 = B.og_pm_longrange(pm, pos, mass, empty)
    assert a0.shape == (0, 3)
    with pytest.raises(B.OgError):
        B.og_pm_create(33, w.L, r_s)
    # og.h: an active_idx entry >= n gets a zero force and is latched in the handle (og_pm_status); the other targets
    # are unaffected
    assert B.og_pm_status(pm) == B.OG_OK
    good = torch.from_numpy(act[:64].view(np.int32)).cuda()
    a_g, p_g = B.og_pm_longrange(pm, pos, mass, good)
    assert B.og_pm_status(pm) == B.OG_OK
    bad = good.clone()
    bad[7] = w.n                                                           # one past the end
    bad[40] = -1                                                           # 0xffffffff
    a_b, p_b = B.og_pm_longrange(pm, pos, mass, bad)
    assert B.og_pm_status(pm) == B.OG_ERR_INVALID_ARG and "active_idx" in B.og_last_error()
    keep = torch.ones(64, dtype=torch.bool, device="cuda")
    keep[7] = keep[40] = False
    # (two PM calls agree to fp32 rounding only: the mass assignment sums with atomics, og.h)
    assert float((a_b[keep] - a_g[keep]).abs().max()) <= 1e-4 * float(a_g.abs().max())
    assert float((p_b[keep] - p_g[keep]).abs().max()) <= 1e-4 * float(p_g.abs().max())
    assert float(a_b[~keep].abs().max()) == 0.0 and float(p_b[~keep].abs().max()) == 0.0
    B.og_pm_longrange(pm, pos, mass, good)
    assert B.og_pm_status(pm) == B.OG_ERR_INVALID_ARG                      # latched until the handle is freed
    B.og_pm_free(pm)


def test_treepm_total_force_is_the_periodic_newtonian_force(B):
    """Short-range walk + PM on the device vs Ewald on the oracle side (= O(N^2) short-range oracle without the hard
    cutoff + exact long-range k-space sum, tests/test_oracle_pm.py): the residual is the TreePM error (mesh, tree
    opening, hard cutoff at 4.5 r_s), a few 1e-3 of the rms force, not a sign / factor / split-scale mistake."""
    import torch
    from test_oracle_pm import _ewald
    rng = np.random.default_rng(11)
    n, L, ng = 400, 1.0, 32
    pos = np.mod(0.5 + 0.12 * rng.standard_normal((n, 3)), L).astype(np.float32)
    mass = ((rng.random(n) + 0.5) / n).astype(np.float32)
    eps = np.full(n, 1e-4, np.float32)
    r_s = 1.25 * L / ng
    dpos, dmass, deps = (torch.from_numpy(x).cuda() for x in (pos, mass, eps))
    tree = B.og_tree_build(dpos, dmass, deps, L, B.make_params(r_s, alpha=0.0005))
    a_s, _ = B.og_shortrange_accel(tree, None, None)
    a_s2, _ = B.og_shortrange_accel(tree, None, torch.linalg.vector_norm(a_s, dim=1).contiguous())
    pm = B.og_pm_create(ng, L, r_s)
    a_l, _ = B.og_pm_longrange(pm, dpos, dmass)
    a_tot = (a_s2 + a_l).cpu().numpy().astype(np.float64)
    B.og_tree_free(tree)
    B.og_pm_free(pm)
    sel = np.arange(0, n, 4)
    a_ew = _ewald(pos, mass, L)[sel]
    arms = np.sqrt((a_ew ** 2).sum(1).mean())
    e = np.linalg.norm(a_tot[sel] - a_ew, axis=1) / arms
    assert np.median(e) < 5e-3 and e.max() < 5e-2, (np.median(e), e.max())
    # and it is the SUM that matches: either part alone is far off
    assert np.median(np.linalg.norm(a_s2.cpu().numpy()[sel] - a_ew, axis=1) / arms) > 0.05
