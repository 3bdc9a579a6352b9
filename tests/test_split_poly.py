"""-m "not gpu": the split-factor approximation of the CUDA path (csrc/walk_math.cuh: E = exp(-w^2) P10(w),
T = E + 2 w / sqrt(pi) exp(-w^2)) meets the R18 budget (abs error <= 1e-6; DESIGN.md Sec. 5.1 states 1.8e-7)
on its whole range w in [0, OG_WMAX], evaluated here in fp32 Horner from the coefficients parsed out of the
header and compared with the exact erfc / exp (math.erfc, fp64) -- the definition the oracle uses."""
import math
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HDR = os.path.join(ROOT, "paper_2606_17145_b200", "csrc", "walk_math.cuh")


def _coefficients():
    src = open(HDR).read()
    body = src[src.index("void og_split("):]
    body = body[:body.index("E = p * ex;")]
    lead = float(re.search(r"float p = ([-+0-9.eE]+)f;", body).group(1))
    rest = [float(x) for x in re.findall(r"p = fmaf\(p, w, ([-+0-9.eE]+)f\);", body)]
    wmax = float(re.search(r"#define OG_WMAX ([0-9.]+)f", src).group(1))
    return [lead] + rest, wmax          # highest degree first


def test_header_polynomial_meets_r18_budget():
    coef, wmax = _coefficients()
    assert len(coef) == 11 and wmax == 2.5
    w = np.linspace(0.0, wmax, 200001).astype(np.float32)
    p = np.full_like(w, np.float32(coef[0]))
    for c in coef[1:]:
        # fmaf: one rounding of p * w + c
        p = (p.astype(np.float64) * w.astype(np.float64) + np.float64(np.float32(c))).astype(np.float32)
    w64 = w.astype(np.float64)
    ex = np.exp(-(w64 * w64)).astype(np.float32)          # ex2.approx is accurate to ~2 ulp: far below the budget
    E = (p.astype(np.float64) * ex).astype(np.float32).astype(np.float64)
    T = (np.float64(np.float32(1.1283791670955126)) * w64 * ex + E).astype(np.float32).astype(np.float64)
    E_ref = np.array([math.erfc(x) for x in w64])
    T_ref = E_ref + 2.0 / math.sqrt(math.pi) * w64 * np.exp(-w64 * w64)
    eE, eT = np.abs(E - E_ref).max(), np.abs(T - T_ref).max()
    assert eE <= 3e-7 and eT <= 3e-7, (eE, eT)
    # exact limits the walk relies on: T(0) = E(0) = 1 to rounding, both decreasing
    assert abs(T[0] - 1.0) <= 2e-7 and abs(E[0] - 1.0) <= 2e-7
    assert np.all(np.diff(T_ref) <= 0)


def test_build_rejects_rcut_beyond_polynomial_range():
    src = open(os.path.join(ROOT, "paper_2606_17145_b200", "csrc", "api.cu")).read()
    assert "rcut_over_rs > 5.0f" in src   # 2 OG_WMAX; the runtime behaviour is checked by tests/test_gpu_edge.py
