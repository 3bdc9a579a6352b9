"""Helpers shared by the -m gpu parity tests: run the CUDA path through the C ABI binding and
the oracle on the same seeded inputs.  The oracle (oracle/) and the CUDA path share no code;
only the seeded generators (paper_2606_17145_b200.workloads) serve both."""
from __future__ import annotations

import numpy as np

import oracle


def oracle_params(w, leaf_max=8, alpha=None, theta=None):
    return oracle.make_params(w.L, w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs,
                              alpha=w.alpha if alpha is None else alpha,
                              theta=w.theta if theta is None else theta, leaf_max=leaf_max)


def gpu_params(w, leaf_max=8, flags=0, alpha=None, theta=None, max_nodes=0, walk_stack_entries=0,
               walk_spill_entries=0):
    from paper_2606_17145_b200 import binding as B
    return B.make_params(w.r_s, G=w.G, rcut_over_rs=w.rcut_over_rs, alpha=w.alpha if alpha is None else alpha,
                         theta=w.theta if theta is None else theta, leaf_max=leaf_max, max_nodes=max_nodes,
                         flags=B.OG_PERIODIC | flags, walk_stack_entries=walk_stack_entries,
                         walk_spill_entries=walk_spill_entries)


def to_dev(w):
    import torch
    dev = torch.device("cuda:0")
    return (torch.from_numpy(w.pos).to(dev), torch.from_numpy(w.mass).to(dev), torch.from_numpy(w.eps).to(dev))


def u64(t):
    """int64-viewed device tensor -> numpy uint64"""
    return t.cpu().numpy().view(np.uint64)


def u32(t):
    return t.cpu().numpy().view(np.uint32)


def rel_err(a_gpu, a_orc):
    """R26: ||a_gpu - a_orc||_2 / ||a_orc||_2 per target."""
    a_gpu = np.asarray(a_gpu, np.float64)
    num = np.linalg.norm(a_gpu - a_orc, axis=1)
    den = np.linalg.norm(a_orc, axis=1)
    ok = den > 0
    return num[ok] / den[ok], int((~ok).sum())


def rel_err_scalar(p_gpu, p_orc):
    p_gpu = np.asarray(p_gpu, np.float64)
    ok = np.abs(p_orc) > 0
    return np.abs(p_gpu[ok] - p_orc[ok]) / np.abs(p_orc[ok])


def check_acc(a_gpu, a_orc, p99=1e-4, mx=1e-2, what=""):
    e, nzero = rel_err(a_gpu, a_orc)
    assert np.all(np.isfinite(a_gpu)), f"{what}: non-finite acceleration"
    q99 = float(np.percentile(e, 99)) if e.size else 0.0
    m = float(e.max()) if e.size else 0.0
    assert q99 <= p99, f"{what}: p99 relative acceleration error {q99:.3e} > {p99}"
    assert m <= mx, f"{what}: max relative acceleration error {m:.3e} > {mx}"
    return q99, m
