"""ctypes binding of libogtree.so (include/og.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels of csrc/.  PyTorch is used for device memory and streams.

There is no CPU fallback: importing this module without the built library raises, and every
compute call fails if no CUDA device is present.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libogtree.so")

# og_status
OG_OK = 0
OG_ERR_INVALID_ARG = -1
OG_ERR_OUT_OF_MEMORY = -2
OG_ERR_NODE_OVERFLOW = -3
OG_ERR_CUDA = -4
OG_ERR_BAD_POSITION = -5
OG_ERR_STACK_OVERFLOW = -6
OG_ERR_NGB_OVERFLOW = -7
# flags
OG_PERIODIC = 1
OG_VALIDATE_POS = 2
OG_COUNT = 4
OG_WALK_G32 = 8
OG_WALK_G8 = 16
# og_field
(OG_F_KEYS_SORTED, OG_F_PERM, OG_F_INV_PERM, OG_F_SPOS, OG_F_SH, OG_F_NODE_LEVEL, OG_F_NODE_FIRST,
 OG_F_NODE_COUNT, OG_F_NODE_FIRST_CHILD, OG_F_NODE_NCHILD, OG_F_NODE_COM, OG_F_NODE_CELL, OG_F_NODE_LO,
 OG_F_NODE_HI, OG_F_LEVEL_START, OG_F_WALK_COST) = range(16)

_FIELD_DTYPE = {
    OG_F_KEYS_SORTED: ("<u8", 8), OG_F_PERM: ("<u4", 4), OG_F_INV_PERM: ("<u4", 4), OG_F_SPOS: ("<f4", 4),
    OG_F_SH: ("<f4", 4), OG_F_NODE_LEVEL: ("|u1", 1), OG_F_NODE_FIRST: ("<u4", 4), OG_F_NODE_COUNT: ("<u4", 4),
    OG_F_NODE_FIRST_CHILD: ("<u4", 4), OG_F_NODE_NCHILD: ("|u1", 1), OG_F_NODE_COM: ("<f4", 4),
    OG_F_NODE_CELL: ("<f4", 4), OG_F_NODE_LO: ("<f4", 4), OG_F_NODE_HI: ("<f4", 4), OG_F_LEVEL_START: ("<u4", 4), OG_F_WALK_COST: ("<u4", 4),
}


class OgError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"og_status {code}: {msg}")
        self.code = code


class og_params(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("flags", C.c_uint32), ("G", C.c_float), ("r_s", C.c_float),
                ("rcut_over_rs", C.c_float), ("alpha", C.c_float), ("theta", C.c_float),
                ("leaf_max", C.c_uint32), ("max_nodes", C.c_uint32), ("walk_stack_entries", C.c_uint32),
                ("walk_spill_entries", C.c_uint32), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t)]


class og_stats(C.Structure):
    _fields_ = [("n", C.c_uint64), ("n_nodes", C.c_uint64), ("max_level", C.c_uint32), ("walk_targets_per_warp", C.c_uint32),
                ("V_full", C.c_uint64), ("V_cull", C.c_uint64), ("A_in", C.c_uint64), ("P_in", C.c_uint64),
                ("P_soft", C.c_uint64), ("P_out", C.c_uint64), ("fp64_rechecks", C.c_uint64),
                ("cl_drop", C.c_uint64), ("cl_open", C.c_uint64), ("cl_accept", C.c_uint64),
                ("cl_generic", C.c_uint64), ("pt_drop", C.c_uint64), ("pt_shift", C.c_uint64),
                ("pt_wrap", C.c_uint64), ("batches", C.c_uint64), ("stack_spills", C.c_uint64)]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_ }


def make_params(r_s, G=1.0, rcut_over_rs=4.5, alpha=0.005, theta=0.5, leaf_max=8, max_nodes=0, flags=OG_PERIODIC,
                walk_stack_entries=0, walk_spill_entries=0) -> og_params:
    return og_params(C.sizeof(og_params), flags | OG_PERIODIC, G, r_s, rcut_over_rs, alpha, theta, leaf_max,
                     max_nodes, walk_stack_entries, walk_spill_entries, None, 0)


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_17145_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, u64, u32p = C.c_void_p, C.c_uint64, C.c_void_p
    lib.og_tree_workspace_bytes.restype = C.c_size_t
    lib.og_tree_workspace_bytes.argtypes = [u64, C.POINTER(og_params)]
    lib.og_tree_build.restype = vp
    lib.og_tree_build.argtypes = [vp, vp, vp, u64, C.c_float, C.POINTER(og_params), vp]
    lib.og_shortrange_accel.restype = C.c_int
    lib.og_shortrange_accel.argtypes = [vp, u32p, u64, vp, vp, vp, vp]
    lib.og_tree_get.restype = C.c_int
    lib.og_tree_get.argtypes = [vp, C.c_int, C.POINTER(vp), C.POINTER(u64)]
    lib.og_tree_status.restype = C.c_int
    lib.og_tree_status.argtypes = [vp]
    lib.og_tree_stats.restype = C.c_int
    lib.og_tree_stats.argtypes = [vp, C.POINTER(og_stats)]
    lib.og_tree_free.restype = None
    lib.og_tree_free.argtypes = [vp, vp]
    lib.og_last_error.restype = C.c_char_p
    lib.og_last_error.argtypes = []
    lib.og_morton_keys.restype = C.c_int
    lib.og_morton_keys.argtypes = [vp, u64, C.c_float, vp, vp, vp]
    lib.og_radix_sort_scratch_bytes.restype = C.c_size_t
    lib.og_radix_sort_scratch_bytes.argtypes = [u64]
    lib.og_radix_sort_pairs.restype = C.c_int
    lib.og_radix_sort_pairs.argtypes = [vp, vp, vp, vp, u64, C.c_int, C.c_int, vp, C.c_size_t,
                                        C.POINTER(C.c_int), vp]
    lib.og_radix_sort_pairs_noalloc.restype = C.c_int
    lib.og_radix_sort_pairs_noalloc.argtypes = [vp, vp, vp, vp, u64, C.c_int, C.c_int, C.POINTER(C.c_int), vp]
    lib.og_shortrange_accel_host.restype = C.c_int
    lib.og_shortrange_accel_host.argtypes = [vp, vp, vp, u64, C.c_float, C.POINTER(og_params), vp, u64, vp, vp,
                                             vp, vp]
    lib.og_trim.restype = C.c_int
    lib.og_trim.argtypes = []
    lib.og_pm_create.restype = vp
    lib.og_pm_create.argtypes = [C.c_uint32, C.c_float, C.c_float, C.c_float, vp]
    lib.og_pm_longrange.restype = C.c_int
    lib.og_pm_longrange.argtypes = [vp, vp, vp, u64, u32p, u64, vp, vp, vp]
    lib.og_pm_free.restype = None
    lib.og_pm_free.argtypes = [vp, vp]
    lib.og_ts_scratch_bytes.restype = C.c_size_t
    lib.og_ts_scratch_bytes.argtypes = [u64]
    lib.og_ts_drift.restype = C.c_int
    lib.og_ts_drift.argtypes = [vp, vp, u64, C.c_float, C.c_float, vp]
    lib.og_ts_next_tick.restype = C.c_int
    lib.og_ts_next_tick.argtypes = [vp, u64, u64, C.c_uint32, C.POINTER(u64), vp, C.c_size_t, vp]
    lib.og_ts_active_list.restype = C.c_int
    lib.og_ts_active_list.argtypes = [vp, u64, u64, C.c_uint32, vp, C.POINTER(u64), vp, C.c_size_t, vp]
    lib.og_shortrange_accel_ext.restype = C.c_int
    lib.og_shortrange_accel_ext.argtypes = [vp, vp, vp, u64, vp, vp, vp, vp]
    lib.og_domain_cell_hist.restype = C.c_int
    lib.og_domain_cell_hist.argtypes = [vp, u64, C.c_float, vp, vp]
    lib.og_domain_owner.restype = C.c_int
    lib.og_domain_owner.argtypes = [vp, u64, C.c_float, vp, C.c_uint32, vp, vp]
    lib.og_let_export_list.restype = C.c_int
    lib.og_let_export_list.argtypes = [vp, u64, vp, C.c_uint32, C.c_float, C.c_float, vp, C.POINTER(C.c_uint64), vp]
    lib.og_let_accumulate.restype = C.c_int
    lib.og_let_accumulate.argtypes = [vp, vp, vp, vp, vp, u64, u64, vp]
    lib.og_sph_density.restype = C.c_int
    lib.og_sph_density.argtypes = [vp, u32p, u64, C.c_float, C.c_float, vp, vp, vp, vp, vp]
    lib.og_ts_kick.restype = C.c_int
    lib.og_ts_kick.argtypes = [vp, vp, vp, u32p, u64, u64, vp, vp, C.c_float, C.c_float, C.c_uint32, u64, C.c_int, vp, vp]
    lib.og_pm_status.restype = C.c_int
    lib.og_pm_status.argtypes = [vp, vp]
    return lib


_lib = _load()

EXPORTS = ("og_tree_workspace_bytes", "og_tree_build", "og_shortrange_accel", "og_tree_get", "og_tree_status",
           "og_tree_stats", "og_tree_free", "og_last_error", "og_morton_keys", "og_radix_sort_scratch_bytes",
           "og_radix_sort_pairs", "og_radix_sort_pairs_noalloc", "og_shortrange_accel_host", "og_trim", "og_pm_create", "og_pm_longrange",
           "og_pm_free", "og_pm_status", "og_ts_scratch_bytes", "og_ts_drift", "og_ts_next_tick", "og_ts_active_list", "og_ts_kick",
           "og_sph_density", "og_shortrange_accel_ext", "og_domain_cell_hist", "og_domain_owner", "og_let_export_list",
           "og_let_accumulate")


def _err() -> str:
    return (_lib.og_last_error() or b"").decode()


def _check(rc: int):
    if rc != OG_OK:
        raise OgError(rc, _err())


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _dev(t: torch.Tensor | None, dtype, name: str):
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of {dtype}, got {t.dtype} on {t.device}")
    return t.data_ptr()


class _DevView:
    """Wraps a raw device pointer for torch.as_tensor (no copy)."""

    def __init__(self, ptr: int, n: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr, "data": (ptr, False), "version": 2}


@dataclass
class Tree:
    handle: int
    n: int
    box: float
    params: og_params
    _keep: tuple = ()

    def __del__(self):
        try:
            og_tree_free(self)
        except Exception:
            pass


def og_tree_workspace_bytes(n: int, params: og_params) -> int:
    return int(_lib.og_tree_workspace_bytes(n, C.byref(params)))


def og_tree_build(pos: torch.Tensor, mass: torch.Tensor, soft: torch.Tensor, box: float, params: og_params,
                  stream=None, workspace: torch.Tensor | None = None) -> Tree:
    """Rows a1..a5.  pos f32 [n][3], mass f32 [n], soft f32 [n]: CUDA tensors (borrowed)."""
    n = int(pos.shape[0])
    p = og_params.from_buffer_copy(params)
    if workspace is not None:
        p.workspace = workspace.data_ptr()
        p.workspace_bytes = workspace.numel() * workspace.element_size()
    h = _lib.og_tree_build(_dev(pos, torch.float32, "pos"), _dev(mass, torch.float32, "mass"),
                           _dev(soft, torch.float32, "soft"), n, float(box), C.byref(p), _stream(stream))
    if not h:
        raise OgError(OG_ERR_INVALID_ARG, _err())
    return Tree(h, n, float(box), p, (workspace,))


def og_shortrange_accel(tree: Tree, active_idx: torch.Tensor | None = None, a_old: torch.Tensor | None = None,
                        want_pot: bool = True, stream=None, acc_out: torch.Tensor | None = None,
                        pot_out: torch.Tensor | None = None):
    """Rows a6..a7.  active_idx: int32/uint32 CUDA tensor of ORIGINAL indices or None (all).
    a_old: f32 CUDA tensor in active order or None (geometric criterion).  -> (acc [na][3], pot [na] | None)"""
    na = tree.n if active_idx is None else int(active_idx.shape[0])
    dev = torch.device("cuda", torch.cuda.current_device())
    if acc_out is None:
        acc_out = torch.empty((na, 3), dtype=torch.float32, device=dev)
    if pot_out is None and want_pot:
        pot_out = torch.empty((na,), dtype=torch.float32, device=dev)
    ai = None
    if active_idx is not None:
        if active_idx.dtype not in (torch.int32, torch.uint32):
            raise TypeError("active_idx must be int32 / uint32")
        if not (active_idx.is_cuda and active_idx.is_contiguous()):
            raise TypeError("active_idx must be a contiguous CUDA tensor")
        ai = active_idx.data_ptr()
    rc = _lib.og_shortrange_accel(tree.handle, ai, na, _dev(a_old, torch.float32, "a_old"),
                                  _dev(acc_out, torch.float32, "acc_out"),
                                  _dev(pot_out, torch.float32, "pot_out"), _stream(stream))
    _check(rc)
    return acc_out, pot_out


def og_tree_get(tree: Tree, field: int) -> torch.Tensor:
    """Device view (no copy) of one tree array; valid until the tree is freed."""
    ptr, cnt = C.c_void_p(), C.c_uint64()
    _check(_lib.og_tree_get(tree.handle, field, C.byref(ptr), C.byref(cnt)))
    typestr, _ = _FIELD_DTYPE[field]
    if cnt.value == 0:
        return torch.empty(0)
    if typestr == "<u8":   # torch has no CUDA uint64 arithmetic; view as int64 (bit pattern preserved)
        typestr = "<i8"
    if typestr == "<u4":
        typestr = "<i4"
    t = torch.as_tensor(_DevView(ptr.value, int(cnt.value), typestr), device="cuda")
    if field in (OG_F_SPOS, OG_F_NODE_COM, OG_F_NODE_CELL, OG_F_NODE_LO, OG_F_NODE_HI):
        t = t.view(-1, 4)
    return t


def og_tree_status(tree: Tree) -> int:
    return int(_lib.og_tree_status(tree.handle))


def og_tree_stats(tree: Tree) -> dict:
    s = og_stats()
    _check(_lib.og_tree_stats(tree.handle, C.byref(s)))
    return s.as_dict()


def og_tree_free(tree: Tree, stream=None):
    if tree.handle:
        h, tree.handle = tree.handle, 0
        _lib.og_tree_free(h, _stream(stream) if torch.cuda.is_available() else None)


def og_last_error() -> str:
    return _err()


def og_morton_keys(pos: torch.Tensor, box: float, stream=None):
    """Row a1.  -> (keys int64-viewed u64 [n], idx int32 [n])"""
    n = int(pos.shape[0])
    keys = torch.empty(n, dtype=torch.int64, device=pos.device)
    idx = torch.empty(n, dtype=torch.int32, device=pos.device)
    _check(_lib.og_morton_keys(_dev(pos, torch.float32, "pos"), n, float(box), keys.data_ptr(), idx.data_ptr(),
                               _stream(stream)))
    return keys, idx


def og_radix_sort_scratch_bytes(n: int) -> int:
    return int(_lib.og_radix_sort_scratch_bytes(n))


def og_radix_sort_pairs(keys: torch.Tensor, vals: torch.Tensor, begin_bit: int = 0, end_bit: int = 64,
                        stream=None):
    """Row a2.  keys int64 (u64 bit pattern), vals int32: sorted IN PLACE or into fresh buffers;
    -> (keys_sorted, vals_sorted).  The inputs are clobbered (ping-pong)."""
    n = int(keys.shape[0])
    k2, v2 = torch.empty_like(keys), torch.empty_like(vals)
    scratch = torch.empty(og_radix_sort_scratch_bytes(n), dtype=torch.uint8, device=keys.device)
    in_alt = C.c_int(0)
    _check(_lib.og_radix_sort_pairs(_dev(keys, torch.int64, "keys"), _dev(vals, torch.int32, "vals"),
                                    k2.data_ptr(), v2.data_ptr(), n, begin_bit, end_bit, scratch.data_ptr(),
                                    scratch.numel(), C.byref(in_alt), _stream(stream)))
    torch.cuda.current_stream().synchronize()  # scratch must outlive the sort
    return (k2, v2) if in_alt.value else (keys, vals)


OG_SORT_NOALLOC_MAX_N = 1 << 20


def og_radix_sort_pairs_noalloc(keys: torch.Tensor, vals: torch.Tensor, keys_alt: torch.Tensor, vals_alt: torch.Tensor,
                                begin_bit: int = 0, end_bit: int = 64, stream=None):
    """Row a2 without any allocation (og.h: og_radix_sort_pairs_noalloc): for callers that own all their device memory
    up front and cannot allocate a per-call scratch.  The caller passes all four ping-pong buffers (keys int64 = u64 bit
    pattern, vals int32, n <= OG_SORT_NOALLOC_MAX_N each); the scratch is the library's built-in array, shared by every
    call on the device, so calls must not overlap on the GPU.  Nothing is allocated here either: the return value is
    the pair of the caller's own tensors that holds the sorted data, (keys_alt, vals_alt) or (keys, vals).  Make the
    first call on a device outside a stream capture (the library resolves the array's address then)."""
    n = int(keys.shape[0])
    if int(vals.shape[0]) != n or int(keys_alt.shape[0]) < n or int(vals_alt.shape[0]) < n:
        raise ValueError("og_radix_sort_pairs_noalloc: vals / keys_alt / vals_alt must hold n elements")
    in_alt = C.c_int(0)
    _check(_lib.og_radix_sort_pairs_noalloc(_dev(keys, torch.int64, "keys"), _dev(vals, torch.int32, "vals"),
                                            _dev(keys_alt, torch.int64, "keys_alt"), _dev(vals_alt, torch.int32, "vals_alt"),
                                            n, begin_bit, end_bit, C.byref(in_alt), _stream(stream)))
    return (keys_alt, vals_alt) if in_alt.value else (keys, vals)


def og_shortrange_accel_host(pos, mass, soft, box: float, params: og_params, active_idx=None, a_old=None,
                             want_pot: bool = True, stream=None, acc_out=None, pot_out=None):
    """End-to-end with HOST tensors (CPU torch tensors, pinned recommended): H2D + build + walk + D2H."""
    n = int(pos.shape[0])
    na = n if active_idx is None else int(active_idx.shape[0])
    for name, t in (("pos", pos), ("mass", mass), ("soft", soft)):
        if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
            raise TypeError(f"{name}: expected a contiguous CPU float32 tensor")
    if acc_out is None:
        acc_out = torch.empty((na, 3), dtype=torch.float32).pin_memory()
    if pot_out is None and want_pot:
        pot_out = torch.empty((na,), dtype=torch.float32).pin_memory()
    p = og_params.from_buffer_copy(params)
    rc = _lib.og_shortrange_accel_host(pos.data_ptr(), mass.data_ptr(), soft.data_ptr(), n, float(box),
                                       C.byref(p), None if active_idx is None else active_idx.data_ptr(), na,
                                       None if a_old is None else a_old.data_ptr(), acc_out.data_ptr(),
                                       None if pot_out is None else pot_out.data_ptr(), _stream(stream))
    _check(rc)
    return acc_out, pot_out


def og_trim():
    """Returns the memory cached in the library's stream-ordered pool to the driver."""
    _check(_lib.og_trim())


# ---- row f1: PM long-range force -------------------------------------------------------------------------
class Pm:
    def __init__(self, handle: int, ng: int, box: float):
        self.handle, self.ng, self.box = handle, ng, box

    def __del__(self):
        try:
            og_pm_free(self)
        except Exception:
            pass


def og_pm_create(ng: int, box: float, r_s: float, G: float = 1.0, stream=None) -> Pm:
    h = _lib.og_pm_create(int(ng), float(box), float(r_s), float(G), _stream(stream))
    if not h:
        raise OgError(OG_ERR_INVALID_ARG, _err())
    return Pm(h, int(ng), float(box))


def og_pm_longrange(pm: Pm, pos: torch.Tensor, mass: torch.Tensor, active_idx: torch.Tensor | None = None,
                    want_pot: bool = True, stream=None):
    """-> (acc [na][3], pot [na] | None): long-range acceleration and potential at the targets."""
    n = int(pos.shape[0])
    na = n if active_idx is None else int(active_idx.shape[0])
    acc = torch.empty((na, 3), dtype=torch.float32, device=pos.device)
    pot = torch.empty((na,), dtype=torch.float32, device=pos.device) if want_pot else None
    ai = None
    if active_idx is not None:
        if active_idx.dtype not in (torch.int32, torch.uint32) or not (active_idx.is_cuda and active_idx.is_contiguous()):
            raise TypeError("active_idx must be a contiguous int32 / uint32 CUDA tensor")
        ai = active_idx.data_ptr()
    _check(_lib.og_pm_longrange(pm.handle, _dev(pos, torch.float32, "pos"), _dev(mass, torch.float32, "mass"), n, ai, na,
                                acc.data_ptr(), None if pot is None else pot.data_ptr(), _stream(stream)))
    return acc, pot


def og_pm_status(pm: Pm, stream=None) -> int:
    """Synchronises the stream; OG_OK, or OG_ERR_INVALID_ARG if an og_pm_longrange on this handle met a bad active index."""
    return int(_lib.og_pm_status(pm.handle, _stream(stream)))


OG_TS_BAD_INDEX = 8


def og_pm_free(pm: Pm, stream=None):
    if pm.handle:
        h, pm.handle = pm.handle, 0
        _lib.og_pm_free(h, _stream(stream) if torch.cuda.is_available() else None)


# ---- row f2: time-step shell ---------------------------------------------------------------------------------
def og_ts_scratch_bytes(n: int) -> int:
    return int(_lib.og_ts_scratch_bytes(n))


def og_ts_drift(pos: torch.Tensor, vel: torch.Tensor, dt: float, box: float, stream=None):
    _check(_lib.og_ts_drift(_dev(pos, torch.float32, "pos"), _dev(vel, torch.float32, "vel"), int(pos.shape[0]), float(dt),
                            float(box), _stream(stream)))


def og_ts_next_tick(bins: torch.Tensor, tick: int, bmax: int, scratch: torch.Tensor, stream=None) -> int:
    out = C.c_uint64(0)
    _check(_lib.og_ts_next_tick(_dev(bins, torch.uint8, "bin"), int(bins.shape[0]), int(tick), int(bmax), C.byref(out),
                                scratch.data_ptr(), scratch.numel() * scratch.element_size(), _stream(stream)))
    return int(out.value)


def og_ts_active_list(bins: torch.Tensor, tick: int, bmax: int, active_idx: torch.Tensor, scratch: torch.Tensor,
                      stream=None) -> int:
    """Fills active_idx (int32 CUDA tensor of >= n elements) with the ascending active particles; -> their number."""
    out = C.c_uint64(0)
    _check(_lib.og_ts_active_list(_dev(bins, torch.uint8, "bin"), int(bins.shape[0]), int(tick), int(bmax),
                                  _dev(active_idx, torch.int32, "active_idx"), C.byref(out), scratch.data_ptr(),
                                  scratch.numel() * scratch.element_size(), _stream(stream)))
    return int(out.value)


def og_ts_kick(vel: torch.Tensor, bins: torch.Tensor, a_old: torch.Tensor, active_idx: torch.Tensor | None, n_active: int,
               acc: torch.Tensor, soft: torch.Tensor, eta: float, dt_max: float, bmax: int, tick: int, first: bool,
               status: torch.Tensor | None = None, stream=None):
    """status: int32 CUDA tensor [1] zeroed by the caller (or None): bit OG_TS_BAD_INDEX is set when an active_idx entry
    is >= n (og.h)."""
    _check(_lib.og_ts_kick(_dev(vel, torch.float32, "vel"), _dev(bins, torch.uint8, "bin"), _dev(a_old, torch.float32, "a_old"),
                           None if active_idx is None else _dev(active_idx, torch.int32, "active_idx"), int(vel.shape[0]),
                           int(n_active), _dev(acc, torch.float32, "acc"), _dev(soft, torch.float32, "soft"), float(eta),
                           float(dt_max), int(bmax), int(tick), 1 if first else 0, _dev(status, torch.int32, "status"),
                           _stream(stream)))


def og_sph_density(tree: Tree, n_des: float, active_idx: torch.Tensor | None = None, h_guess: torch.Tensor | None = None,
                   tol_n: float = 0.0, want_rho: bool = True, want_nn: bool = True, stream=None):
    """Row f3.  -> (h [na], rho [na] | None, N [na] | None) in the caller's order."""
    na = tree.n if active_idx is None else int(active_idx.shape[0])
    dev = torch.device("cuda", torch.cuda.current_device())
    h = torch.empty(na, dtype=torch.float32, device=dev)
    rho = torch.empty(na, dtype=torch.float32, device=dev) if want_rho else None
    nn = torch.empty(na, dtype=torch.float32, device=dev) if want_nn else None
    _check(_lib.og_sph_density(tree.handle, None if active_idx is None else _dev(active_idx, torch.int32, "active_idx"), na,
                               float(n_des), float(tol_n), _dev(h_guess, torch.float32, "h_guess"),
                               _dev(h, torch.float32, "h_out"), _dev(rho, torch.float32, "rho_out"),
                               _dev(nn, torch.float32, "nn_out"), _stream(stream)))
    return h, rho, nn


# ---- row f4 ----------------------------------------------------------------------------------------------------------
def og_shortrange_accel_ext(tree: Tree, tpos: torch.Tensor, tsoft: torch.Tensor, a_old: torch.Tensor | None,
                            want_pot: bool = True, stream=None):
    """Walk of `tree` for targets that are not its particles.  -> (acc [n_t][3], pot [n_t] | None)"""
    nt = int(tpos.shape[0])
    dev = tpos.device
    acc = torch.empty((nt, 3), dtype=torch.float32, device=dev)
    pot = torch.empty(nt, dtype=torch.float32, device=dev) if want_pot else None
    _check(_lib.og_shortrange_accel_ext(tree.handle, _dev(tpos, torch.float32, "tpos"), _dev(tsoft, torch.float32, "tsoft"), nt,
                                        _dev(a_old, torch.float32, "a_old"), _dev(acc, torch.float32, "acc_out"),
                                        _dev(pot, torch.float32, "pot_out"), _stream(stream)))
    return acc, pot


def og_domain_cell_hist(pos: torch.Tensor, box: float, stream=None) -> torch.Tensor:
    hist = torch.empty(1 << 15, dtype=torch.int32, device=pos.device)
    _check(_lib.og_domain_cell_hist(_dev(pos, torch.float32, "pos"), int(pos.shape[0]), float(box),
                                    _dev(hist, torch.int32, "hist"), _stream(stream)))
    return hist


def og_domain_owner(pos: torch.Tensor, box: float, splitters: torch.Tensor, stream=None) -> torch.Tensor:
    owner = torch.empty(int(pos.shape[0]), dtype=torch.int32, device=pos.device)
    _check(_lib.og_domain_owner(_dev(pos, torch.float32, "pos"), int(pos.shape[0]), float(box),
                                _dev(splitters, torch.int32, "splitters"), int(splitters.shape[0]) - 1,
                                _dev(owner, torch.int32, "owner"), _stream(stream)))
    return owner


def og_let_export_list(tpos: torch.Tensor, boxes: torch.Tensor, r_cut: float, box: float, stream=None) -> torch.Tensor:
    """-> ascending int32 positions of the targets within r_cut of one of the boxes [nb][6]."""
    nt = int(tpos.shape[0])
    out = torch.empty(max(nt, 1), dtype=torch.int32, device=tpos.device)
    cnt = C.c_uint64(0)
    _check(_lib.og_let_export_list(_dev(tpos, torch.float32, "tpos"), nt, _dev(boxes, torch.float32, "boxes"),
                                   int(boxes.shape[0]), float(r_cut), float(box), _dev(out, torch.int32, "list_out"),
                                   C.byref(cnt), _stream(stream)))
    return out[:int(cnt.value)]


def og_let_accumulate(acc: torch.Tensor, pot: torch.Tensor | None, idx: torch.Tensor, part_acc: torch.Tensor,
                      part_pot: torch.Tensor | None, stream=None):
    _check(_lib.og_let_accumulate(_dev(acc, torch.float32, "acc"), _dev(pot, torch.float32, "pot"), _dev(idx, torch.int32, "idx"),
                                  _dev(part_acc, torch.float32, "part_acc"), _dev(part_pot, torch.float32, "part_pot"),
                                  int(idx.shape[0]), int(acc.shape[0]), _stream(stream)))
