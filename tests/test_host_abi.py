"""-m "not gpu": the C-ABI library loads and exports every symbol include/og.h declares; host-side
argument checks work without a device; there is no CPU fallback (compute calls fail loudly)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2606_17145_b200 import build
    build.build()
    from paper_2606_17145_b200 import binding
    return binding


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "og.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(og_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported(B):
    names = _declared_symbols()
    assert "og_tree_build" in names and "og_shortrange_accel" in names
    lib = C.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in og.h but not exported"
    assert set(B.EXPORTS) == set(names)


def test_only_the_documented_calls_are_exported(B):
    """nm -D: the og_* symbols of libogtree.so are exactly the calls og.h declares (no bench / debug helpers)."""
    import subprocess
    out = subprocess.run(["nm", "-D", "--defined-only", B.LIB_PATH], capture_output=True, text=True, check=True).stdout
    exported = sorted(set(re.findall(r"\b(og_[a-z0-9_]+)\b", out)))
    assert exported == _declared_symbols(), exported


def test_params_struct_matches_header(B):
    p = B.make_params(0.01)
    assert p.struct_size == C.sizeof(B.og_params)
    # uint32 x2, float x5, uint32 x4, (4 bytes padding), pointer, size_t
    assert C.sizeof(B.og_params) == 48 + 8 + 8


def test_workspace_bytes_is_host_only(B):
    p = B.make_params(0.01)
    n = 1 << 20
    w = B._lib.og_tree_workspace_bytes(n, C.byref(p))
    assert w > n * (8 + 8 + 4 + 4 + 16 + 4 + 4)      # keys ping-pong, idx ping-pong, spos, sh, inv_perm at least
    bad = B.make_params(0.01)
    bad.struct_size = 4
    assert B._lib.og_tree_workspace_bytes(n, C.byref(bad)) == 0
    assert B._lib.og_tree_workspace_bytes(0, C.byref(p)) == 0


def test_argument_errors_and_no_cpu_fallback(B):
    import torch
    p = B.make_params(0.3)          # r_cut = 1.35 >= box / 2 for box = 1
    t = B._lib.og_tree_build(None, None, None, 16, C.c_float(1.0), C.byref(p), None)
    assert not t
    assert b"r_cut" in B._lib.og_last_error()
    p = B.make_params(0.01)
    t = B._lib.og_tree_build(None, None, None, 16, C.c_float(1.0), C.byref(p), None)
    assert not t and b"non-NULL" in B._lib.og_last_error()
    if not torch.cuda.is_available():
        # a syntactically valid call must fail loudly without a device: nothing computes on the CPU
        buf = (C.c_float * 64)()
        t = B._lib.og_tree_build(buf, buf, buf, 16, C.c_float(1.0), C.byref(p), None)
        assert not t and b"no CUDA device" in B._lib.og_last_error()
    assert B._lib.og_shortrange_accel(None, None, 0, None, None, None, None) == B.OG_ERR_INVALID_ARG
    # the two grouping flags of the walk exclude each other (og.h)
    p = B.make_params(0.01, flags=B.OG_PERIODIC | B.OG_WALK_G8 | B.OG_WALK_G32)
    t = B._lib.og_tree_build(None, None, None, 16, C.c_float(1.0), C.byref(p), None)
    assert not t and b"OG_WALK_G32" in B._lib.og_last_error()


def test_new_rows_reject_bad_arguments_without_a_device(B):
    """Rows f3 / f4: NULL handles and out-of-range scalars are refused on the host before anything is enqueued."""
    L = B._lib
    assert L.og_sph_density(None, None, 10, C.c_float(32.0), C.c_float(0.0), None, None, None, None, None) == B.OG_ERR_INVALID_ARG
    assert b"tree is NULL" in L.og_last_error()
    assert L.og_shortrange_accel_ext(None, None, None, 10, None, None, None, None) == B.OG_ERR_INVALID_ARG
    assert L.og_domain_cell_hist(None, 10, C.c_float(1.0), None, None) == B.OG_ERR_INVALID_ARG
    assert L.og_domain_owner(None, 10, C.c_float(1.0), None, 4, None, None) == B.OG_ERR_INVALID_ARG
    cnt = C.c_uint64(7)
    assert L.og_let_export_list(None, 0, None, 0, C.c_float(0.1), C.c_float(1.0), None, C.byref(cnt), None) == B.OG_OK
    assert cnt.value == 0                                                   # empty input: a no-op that reports 0
    assert L.og_let_export_list(None, 5, None, 3, C.c_float(0.1), C.c_float(1.0), None, C.byref(cnt), None) == B.OG_ERR_INVALID_ARG
    assert L.og_let_accumulate(None, None, None, None, None, 5, 5, None) == B.OG_ERR_INVALID_ARG
    assert L.og_let_accumulate(None, None, None, None, None, 0, 5, None) == B.OG_OK


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_17145_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                s = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import oracle|from oracle)", s, flags=re.M), f
                assert "liboracle" not in s and "oracle.c" not in s, f
