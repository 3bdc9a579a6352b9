"""-m gpu: rows f3 and f4 at BASELINE.json's FULL size (nfw256, 16.8 M particles), in the launch configuration bench.py
times, on SAMPLED outputs the oracle computes one by one (the oracle's cost per target is milliseconds to seconds here).
 * f3: og_sph_density for ALL particles (bench.py --sph), compared on a seeded sample with oracle/sph.py; every
   returned N within 1e-4 n_des of n_des, every h finite and positive (properties that hold at any size).
 * f4: the decomposed pipeline (bench.py --scaling let --let-domains 4) for ALL targets, compared on a seeded sample
   with oracle.let.let_walk (the oracle builds the four domain trees in full and walks only the sample); owners of ALL
   particles bit-exact.
The measured numbers are appended to gpurun_out/full_parity.txt."""
import os
import time

import numpy as np
import pytest

import oracle
from oracle import let as olet
from oracle import sph as osph
from paper_2606_17145_b200 import workloads as W
from gpu_common import gpu_params, oracle_params, rel_err, rel_err_scalar, to_dev

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B(cuda_device):
    from paper_2606_17145_b200 import binding
    return binding


def _log(line):
    print(line)
    try:
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        with open(os.path.join(ROOT, "gpurun_out", "full_parity.txt"), "a") as f:
            f.write(line + "\n")
    except OSError:
        pass


def test_f3_sph_density_full_size_sampled(B):
    import torch
    w = W.make("nfw256")
    n_des = 32.0
    pos, mass, eps = to_dev(w)
    tree = B.og_tree_build(pos, mass, eps, w.L, gpu_params(w))
    h, rho, nn = B.og_sph_density(tree, n_des)
    hw, rhow, _ = B.og_sph_density(tree, n_des, h_guess=h.clone())           # warm start: the same roots
    torch.cuda.synchronize()
    assert B.og_tree_status(tree) == B.OG_OK, B.og_last_error()
    hh, rr, nnn = h.cpu().numpy().astype(np.float64), rho.cpu().numpy().astype(np.float64), nn.cpu().numpy()
    assert np.all(np.isfinite(hh)) and hh.min() > 0 and np.all(np.isfinite(rr)) and rr.min() > 0
    assert np.abs(nnn - n_des).max() <= 1e-4 * n_des                          # every target reached its root
    assert float(((hw - h).abs() / h).max()) <= 2e-6 and float(((rhow - rho).abs() / rho).max()) <= 2e-5
    rng = np.random.default_rng(260617)
    t = np.sort(rng.choice(w.n, size=600, replace=False))
    t0 = time.time()
    ho, ro, no = osph.sph_density(w.pos.astype(np.float64), w.mass.astype(np.float64), w.L, n_des, targets=t)
    sec = time.time() - t0
    eh, er = np.abs(hh[t] - ho) / ho, np.abs(rr[t] - ro) / ro
    _log(f"nfw256           f3 sph     targets {len(t):10d}  h p99 {np.percentile(eh, 99):.2e} max {eh.max():.2e}  rho p99 "
         f"{np.percentile(er, 99):.2e} max {er.max():.2e}  max |N - n_des| over all 16.8 M {np.abs(nnn - n_des).max():.2e}  oracle {sec:.0f} s")
    assert np.percentile(eh, 99) <= 5e-6 and eh.max() <= 1e-4
    assert np.percentile(er, 99) <= 2e-5 and er.max() <= 3e-4
    B.og_tree_free(tree)


def test_f4_let_pipeline_full_size_sampled(B):
    import torch
    from paper_2606_17145_b200 import let
    w = W.make("nfw256")
    R = 4
    prm_o = oracle_params(w)
    dev = torch.device("cuda:0")
    ex = let.LocalExchange(R)

    def parts(a_pp):
        out = {}
        for r in range(R):
            sel = np.arange(r, w.n, R)
            out[r] = let.Domain(*(torch.from_numpy(x[sel]).to(dev) for x in (w.pos, w.mass, w.eps)),
                                torch.from_numpy(sel.astype(np.int64)).to(dev), torch.ones(len(sel), dtype=torch.bool, device=dev),
                                None if a_pp is None else a_pp[torch.from_numpy(sel).to(dev)].contiguous())
        return out

    # a_old for EVERY target from the device's own geometric pipeline pass (the inputs of both sides are the same
    # fp32 numbers, R23; the geometric pass itself is compared on the sample below)
    doms, S = let.decompose(B, parts(None), ex, w.L)
    res, _ = let.let_forces(B, doms, ex, w.L, gpu_params(w), geometric=True, want_pot=False)
    a_pp = torch.zeros(w.n, device=dev)
    a_geo = np.zeros((w.n, 3), np.float32)
    for r in range(R):
        g = doms[r].gid[doms[r].active.long()]
        a_pp[g] = torch.linalg.vector_norm(res[r][0], dim=1)
        a_geo[g.cpu().numpy()] = res[r][0].cpu().numpy()
    doms, S = let.decompose(B, parts(a_pp), ex, w.L)
    res, info = let.let_forces(B, doms, ex, w.L, gpu_params(w))
    acc = np.zeros((w.n, 3), np.float32)
    pot = np.zeros(w.n, np.float32)
    owner_gpu = np.empty(w.n, np.int32)
    for r in range(R):
        g = doms[r].gid[doms[r].active.long()].cpu().numpy()
        acc[g] = res[r][0].cpu().numpy()
        pot[g] = res[r][1].cpu().numpy()
        owner_gpu[doms[r].gid.cpu().numpy()] = r
    # oracle: same decomposition (all particles), walks of a seeded sample of targets
    rng = np.random.default_rng(1714)
    t = np.sort(rng.choice(w.n, size=8192, replace=False)).astype(np.uint32)
    a_old = a_pp.cpu().numpy()
    t0 = time.time()
    a_g, _, oinfo = olet.let_walk(w.pos, w.mass, w.eps, prm_o, R, active_idx=t, a_old=None)
    a_r, p_r, _ = olet.let_walk(w.pos, w.mass, w.eps, prm_o, R, active_idx=t, a_old=a_old[t])
    sec = time.time() - t0
    assert np.array_equal(S, oinfo["splitters"]) and np.array_equal(owner_gpu, oinfo["owner"])
    eg, _ = rel_err(a_geo[t], a_g)
    er, _ = rel_err(acc[t], a_r)
    ep = rel_err_scalar(pot[t], p_r)
    _log(f"nfw256           f4 let R=4 targets {len(t):10d}  acc p99 {np.percentile(er, 99):.2e} max {er.max():.2e} n(>1e-4) "
         f"{int((er > 1e-4).sum())}  geometric pass max {eg.max():.2e}  pot p99 {np.percentile(ep, 99):.2e} max {ep.max():.2e}  "
         f"exported copies {sum(info['n_exported'].values())}  oracle {sec:.0f} s")
    assert np.percentile(er, 99) <= 1e-4 and er.max() <= 1e-2
    assert np.percentile(eg, 99) <= 1e-4 and eg.max() <= 1e-2
    assert np.percentile(ep, 99) <= 1e-4 and ep.max() <= 1e-2
