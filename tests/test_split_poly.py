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
    defs = {int(k): float(v) for k, v in re.findall(r"#define OG_SP(\d+) ([-+0-9.eE]+)f", src)}
    coef = [defs[k] for k in range(max(defs), -1, -1)]          # highest degree first
    assert max(defs) == 10
    # the scalar evaluator is the plain Horner chain over exactly these coefficients ...
    body = src[src.index("void og_split("):]
    body = body[:body.index("\n}\n")]
    assert "float p = OG_SP10;" in body
    pos = 0
    for k in range(9, -1, -1):
        pos = body.index("p = fmaf(p, w, OG_SP%d);" % k, pos)
    # ... and the packed one the even / odd split in w^2 over the same coefficients
    body = src[src.index("void og_split2("):]
    body = body[:body.index("\n}\n")]
    assert "f32x2 pe = bc2(OG_SP10), po = bc2(OG_SP9);" in body
    pos = 0
    for k in range(8, -1, -1):
        pos = body.index("%s = fma2(%s, w2, bc2(OG_SP%d));" % (("pe", "pe", k) if k % 2 == 0 else ("po", "po", k)), pos)
    assert "const f32x2 p = fma2(po, w, pe);" in body
    assert float(re.search(r"#define OG_TWO_OVER_SQRTPI ([0-9.]+)f", src).group(1)) == 1.1283791670955126
    wmax = float(re.search(r"#define OG_WMAX ([0-9.]+)f", src).group(1))
    return coef, wmax


def _fma32(a, b, c):
    """fmaf on float32 arrays: one rounding of a * b + c (the product of two fp32 values is exact in fp64)"""
    return (a.astype(np.float64) * b.astype(np.float64) + np.asarray(c, np.float32).astype(np.float64)).astype(np.float32)


def _check(p, w):
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


def test_header_polynomial_meets_r18_budget():
    """og_split: Horner in fp32."""
    coef, wmax = _coefficients()
    assert len(coef) == 11 and wmax == 2.5
    w = np.linspace(0.0, wmax, 200001).astype(np.float32)
    p = np.full_like(w, np.float32(coef[0]))
    for c in coef[1:]:
        p = _fma32(p, w, c)
    _check(p, w)


def test_header_polynomial_even_odd_order_meets_r18_budget():
    """og_split2 (the packed evaluator of the group walk): even / odd parts in w^2, fp32."""
    coef, wmax = _coefficients()
    c = coef[::-1]                                          # c[k] = coefficient of w^k
    w = np.linspace(0.0, wmax, 200001).astype(np.float32)
    w2 = (w.astype(np.float64) * w.astype(np.float64)).astype(np.float32)
    pe = np.full_like(w, np.float32(c[10]))
    po = np.full_like(w, np.float32(c[9]))
    for k in (8, 6, 4, 2, 0):
        pe = _fma32(pe, w2, c[k])
    for k in (7, 5, 3, 1):
        po = _fma32(po, w2, c[k])
    _check(_fma32(po, w, pe), w)


def test_build_rejects_rcut_beyond_polynomial_range():
    src = open(os.path.join(ROOT, "paper_2606_17145_b200", "csrc", "api.cu")).read()
    assert "rcut_over_rs > 5.0f" in src   # 2 OG_WMAX; the runtime behaviour is checked by tests/test_gpu_edge.py
