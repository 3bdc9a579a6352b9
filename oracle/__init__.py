"""oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes front end of ``oracle/oracle.c``: the plain fp64 CPU restatement of the
TreePM short-range gravity path.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2606_17145_b200`` and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

NCOUNT = 12
COUNTER_NAMES = ("V_full", "V_cull", "A_in", "A_out", "P_in", "P_out", "P_soft", "O_int", "O_leaf",
                 "C_open", "L_open", "self")

# Algorithmic-flop weights of SURVEY.md Sec. 8.4 (frozen here; DESIGN.md prints the table).
FLOP_WEIGHTS = {"V_cull": 6, "V_full": 16, "A_in": 21, "P_out": 11, "P_in": 32, "P_soft_extra": 13}
FLOP_WEIGHTS_NOPOT = {"V_cull": 6, "V_full": 16, "A_in": 16, "P_out": 11, "P_in": 27, "P_soft_extra": 7}


def build(force: bool = False) -> str:
    """Compile oracle.c -> liboracle.so (gcc, -ffp-contract=off, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
               "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class Params(C.Structure):
    _fields_ = [("G", C.c_float), ("L", C.c_float), ("r_s", C.c_float),
                ("rcut_over_rs", C.c_float), ("alpha", C.c_float), ("theta", C.c_float),
                ("leaf_max", C.c_uint32), ("want_pot", C.c_uint32)]


def make_params(L, r_s, G=1.0, rcut_over_rs=4.5, alpha=0.005, theta=0.5, leaf_max=8) -> Params:
    return Params(G, L, r_s, rcut_over_rs, alpha, theta, leaf_max, 1)


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_spline_g.restype = C.c_double
        _lib.orc_spline_g.argtypes = [C.c_double, C.c_double]
        _lib.orc_spline_p.restype = C.c_double
        _lib.orc_spline_p.argtypes = [C.c_double, C.c_double]
        _lib.orc_split_T.restype = C.c_double
        _lib.orc_split_T.argtypes = [C.c_double]
        _lib.orc_split_E.restype = C.c_double
        _lib.orc_split_E.argtypes = [C.c_double]
        _lib.orc_interleave.restype = C.c_uint64
        _lib.orc_interleave.argtypes = [C.c_uint32] * 3
        _lib.orc_tree_build.restype = C.c_int64
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a, ctype=None):
    if a is None:
        return None
    return a.ctypes.data_as(C.c_void_p)


def _c(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a


def num_threads() -> int:
    return int(lib().orc_num_threads())


# ---- scalar kernels (C5) ---------------------------------------------------
def spline_g(r, h):
    return lib().orc_spline_g(float(r), float(h))


def spline_p(r, h):
    return lib().orc_spline_p(float(r), float(h))


def split_T(w):
    return lib().orc_split_T(float(w))


def split_E(w):
    return lib().orc_split_E(float(w))


def pair_eval(params: Params, x, h_i, xj, mj, h_j):
    """Force and potential on a target at x from one source (C5). -> (kind, acc[3], pot)"""
    x = (C.c_double * 3)(*[float(v) for v in x])
    xj = (C.c_double * 3)(*[float(v) for v in xj])
    acc = (C.c_double * 3)()
    pot = C.c_double(0.0)
    f = lib().orc_pair_eval
    f.restype = C.c_int
    f.argtypes = [C.POINTER(Params), C.c_double * 3, C.c_double, C.c_double * 3, C.c_double,
                  C.c_double, C.c_double * 3, C.POINTER(C.c_double)]
    kind = f(C.byref(params), x, float(h_i), xj, float(mj), float(h_j), acc, C.byref(pot))
    return kind, np.array(acc[:]), pot.value


# ---- C1 keys, C2 sort ------------------------------------------------------
def interleave(qx, qy, qz) -> int:
    return int(lib().orc_interleave(int(qx), int(qy), int(qz)))


def deinterleave(key):
    qx, qy, qz = C.c_uint32(), C.c_uint32(), C.c_uint32()
    lib().orc_deinterleave(C.c_uint64(int(key)), C.byref(qx), C.byref(qy), C.byref(qz))
    return qx.value, qy.value, qz.value


def keys(pos: np.ndarray, L: float) -> np.ndarray:
    pos = _c(pos, np.float32)
    n = pos.shape[0]
    out = np.empty(n, dtype=np.uint64)
    lib().orc_keys(_p(pos), C.c_uint64(n), C.c_float(L), _p(out))
    return out


def sort(k: np.ndarray):
    """-> (perm u32[N], keys_sorted u64[N]); ascending (key, original index)."""
    k = _c(k, np.uint64)
    n = k.shape[0]
    perm = np.empty(n, dtype=np.uint32)
    ks = np.empty(n, dtype=np.uint64)
    rc = lib().orc_sort(_p(k), C.c_uint64(n), _p(perm), _p(ks))
    if rc != 0:
        raise MemoryError("orc_sort")
    return perm, ks


# ---- C3 tree, C4 upward ----------------------------------------------------
@dataclass
class Tree:
    """Canonical octree + fp32 node records (R9) + sorted particle copies."""
    n: int
    L: float
    params: Params
    perm: np.ndarray
    inv_perm: np.ndarray
    keys: np.ndarray           # unsorted keys (original order)
    keys_sorted: np.ndarray
    level: np.ndarray
    first: np.ndarray
    count: np.ndarray
    first_child: np.ndarray
    n_child: np.ndarray
    M64: np.ndarray
    s64: np.ndarray
    M: np.ndarray
    s: np.ndarray
    c: np.ndarray
    l: np.ndarray
    hmax: np.ndarray
    lo: np.ndarray
    hi: np.ndarray
    spos: np.ndarray
    smass: np.ndarray
    sh: np.ndarray
    extra: dict = field(default_factory=dict)

    @property
    def n_nodes(self) -> int:
        return int(self.level.shape[0])


def tree_topology(keys_sorted: np.ndarray, leaf_max: int):
    ks = _c(keys_sorted, np.uint64)
    n = ks.shape[0]
    f = lib().orc_tree_build
    nn = f(_p(ks), C.c_uint64(n), C.c_uint32(leaf_max), C.c_int64(0), None, None, None, None, None)
    level = np.empty(nn, np.uint8)
    first = np.empty(nn, np.uint32)
    count = np.empty(nn, np.uint32)
    first_child = np.empty(nn, np.uint32)
    n_child = np.empty(nn, np.uint8)
    nn2 = f(_p(ks), C.c_uint64(n), C.c_uint32(leaf_max), C.c_int64(nn), _p(level), _p(first),
            _p(count), _p(first_child), _p(n_child))
    assert nn2 == nn
    return level, first, count, first_child, n_child


def particle_h(eps: np.ndarray) -> np.ndarray:
    eps = _c(eps, np.float32)
    h = np.empty_like(eps)
    lib().orc_particle_h(_p(eps), C.c_uint64(eps.shape[0]), _p(h))
    return h


def build_tree(pos, mass, eps, params: Params) -> Tree:
    """C1..C4: keys -> sort -> canonical octree -> upward pass."""
    pos = _c(pos, np.float32)
    mass = _c(mass, np.float32)
    eps = _c(eps, np.float32)
    n = pos.shape[0]
    L = float(params.L)
    k = keys(pos, L)
    perm, ks = sort(k)
    inv = np.empty(n, np.uint32)
    inv[perm] = np.arange(n, dtype=np.uint32)
    level, first, count, first_child, n_child = tree_topology(ks, int(params.leaf_max))
    nn = level.shape[0]
    spos = np.ascontiguousarray(pos[perm])
    smass = np.ascontiguousarray(mass[perm])
    sh = particle_h(np.ascontiguousarray(eps[perm]))
    M64 = np.empty(nn, np.float64)
    s64 = np.empty((nn, 3), np.float64)
    M = np.empty(nn, np.float32)
    s = np.empty((nn, 3), np.float32)
    c = np.empty((nn, 3), np.float32)
    l = np.empty(nn, np.float32)
    hmax = np.empty(nn, np.float32)
    lo = np.empty((nn, 3), np.float32)
    hi = np.empty((nn, 3), np.float32)
    rc = lib().orc_upward(_p(ks), _p(spos), _p(smass), _p(sh), C.c_float(L), C.c_int64(nn),
                          _p(level), _p(first), _p(count), _p(first_child), _p(n_child),
                          _p(M64), _p(s64), _p(M), _p(s), _p(c), _p(l), _p(hmax), _p(lo), _p(hi))
    if rc != 0:
        raise MemoryError("orc_upward")
    return Tree(n, L, params, perm, inv, k, ks, level, first, count, first_child, n_child,
                M64, s64, M, s, c, l, hmax, lo, hi, spos, smass, sh)


# ---- C6 walk, C7 direct ----------------------------------------------------
def walk(tree: Tree, active_idx=None, a_old=None, params: Params | None = None,
         want_counters: bool = True):
    """Per-target tree walk.  active_idx: ORIGINAL particle indices (None -> all, identity).
    a_old: fp32 |a| per target in active order, or None -> geometric theta criterion.
    -> acc f64[n_t][3], pot f64[n_t], counters u64[n_t][9]"""
    prm = params if params is not None else tree.params
    if active_idx is None:
        active_idx = np.arange(tree.n, dtype=np.uint32)
    active_idx = _c(active_idx, np.uint32)
    slots = np.ascontiguousarray(tree.inv_perm[active_idx])
    nt = slots.shape[0]
    if a_old is not None:
        a_old = _c(a_old, np.float32)
        assert a_old.shape[0] == nt
    acc = np.zeros((nt, 3), np.float64)
    pot = np.zeros(nt, np.float64)
    cnt = np.zeros((nt, NCOUNT), np.uint64) if want_counters else None
    lib().orc_walk(C.byref(prm), C.c_uint64(nt), _p(slots), _p(a_old), _p(tree.n_child),
                   _p(tree.first), _p(tree.count), _p(tree.first_child), _p(tree.M), _p(tree.s),
                   _p(tree.c), _p(tree.l), _p(tree.hmax), _p(tree.lo), _p(tree.hi),
                   _p(tree.spos), _p(tree.smass), _p(tree.sh), _p(acc), _p(pot), _p(cnt))
    return acc, pot, cnt


def direct(pos, mass, eps, params: Params, target_idx=None):
    """O(N^2) direct short-range sum (C7). -> acc f64[n_t][3], pot f64[n_t]"""
    pos = _c(pos, np.float32)
    mass = _c(mass, np.float32)
    h = particle_h(_c(eps, np.float32))
    n = pos.shape[0]
    if target_idx is not None:
        target_idx = _c(target_idx, np.uint32)
        nt = target_idx.shape[0]
    else:
        nt = n
    acc = np.zeros((nt, 3), np.float64)
    pot = np.zeros(nt, np.float64)
    lib().orc_direct(C.byref(params), C.c_uint64(n), _p(pos), _p(mass), _p(h), C.c_uint64(nt),
                     _p(target_idx), _p(acc), _p(pot))
    return acc, pot


def walk_ext(tree: Tree, tpos, th, a_old=None, params: Params | None = None, want_counters: bool = False):
    """Row f4: the walk of `tree` for targets that are not its particles (imported from another domain): tpos f32[n_t][3],
    th f32[n_t] (= 2.8 eps of the target), a_old f32[n_t] or None.  Nothing is excluded.  -> acc, pot, counters"""
    prm = params if params is not None else tree.params
    tpos = _c(tpos, np.float32)
    th = _c(th, np.float32)
    nt = tpos.shape[0]
    if a_old is not None:
        a_old = _c(a_old, np.float32)
        assert a_old.shape[0] == nt
    acc = np.zeros((nt, 3), np.float64)
    pot = np.zeros(nt, np.float64)
    cnt = np.zeros((nt, NCOUNT), np.uint64) if want_counters else None
    lib().orc_walk_ext(C.byref(prm), C.c_uint64(nt), _p(tpos), _p(th), _p(a_old), _p(tree.n_child),
                       _p(tree.first), _p(tree.count), _p(tree.first_child), _p(tree.M), _p(tree.s),
                       _p(tree.c), _p(tree.l), _p(tree.hmax), _p(tree.lo), _p(tree.hi),
                       _p(tree.spos), _p(tree.smass), _p(tree.sh), _p(acc), _p(pot), _p(cnt))
    return acc, pot, cnt


def direct_ext(pos, mass, eps, params: Params, tpos, teps):
    """O(N n_t) direct short-range sum on targets that are not among the sources. -> acc, pot"""
    pos = _c(pos, np.float32)
    mass = _c(mass, np.float32)
    h = particle_h(_c(eps, np.float32))
    tpos = _c(tpos, np.float32)
    th = particle_h(_c(teps, np.float32))
    nt = tpos.shape[0]
    acc = np.zeros((nt, 3), np.float64)
    pot = np.zeros(nt, np.float64)
    lib().orc_direct_ext(C.byref(params), C.c_uint64(pos.shape[0]), _p(pos), _p(mass), _p(h), C.c_uint64(nt),
                         _p(tpos), _p(th), _p(acc), _p(pot))
    return acc, pot


def algorithmic_flops(counters: np.ndarray, with_pot: bool = True) -> np.ndarray:
    """F_alg per target from the walk counters (SURVEY.md Sec. 8.4 weights).
    -> (F_alg, F_int) arrays; F_int = interaction-only part (last four terms)."""
    w = FLOP_WEIGHTS if with_pot else FLOP_WEIGHTS_NOPOT
    c = counters.astype(np.float64)
    V_full, V_cull, A_in, P_in, P_out, P_soft = c[:, 0], c[:, 1], c[:, 2], c[:, 4], c[:, 5], c[:, 6]
    F_int = w["A_in"] * A_in + w["P_out"] * P_out + w["P_in"] * P_in + w["P_soft_extra"] * P_soft
    F_dec = w["V_cull"] * V_cull + w["V_full"] * V_full
    return F_dec + F_int, F_int
