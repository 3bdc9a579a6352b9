"""og_radix_sort_pairs_noalloc: the radix sort for callers that cannot allocate device memory.

Some users of the library cannot call cudaMalloc when they need a sort: a simulation code that took the whole device
for its own arena at start-up, a step running where an allocation would stall the device or wait on a lock another
thread holds, a component that is only lent buffers.  og_radix_sort_pairs wants a scratch buffer sized per call; the
no-alloc variant keeps that scratch in a fixed array inside libogtree.so (about 4 MiB per GPU, n <= 2^20 pairs) and
allocates nothing.  It must return exactly what the existing path returns (integer work: bit for bit), also on a
second call that finds the first call's leftovers in the shared array, and it must refuse sizes above its limit with
a message that names the limit.

The file name sorts after every other test file on purpose: pytest -x stops at the first failure, so a failure here
must not hide the tests of the main path.  The GPU test stands alone (fresh process) and also runs after the others.
"""
import ctypes as C

import numpy as np
import pytest


@pytest.fixture(scope="module")
def B():
    from paper_2606_17145_b200 import build
    build.build()
    from paper_2606_17145_b200 import binding
    return binding


def test_noalloc_sort_rejects_sizes_beyond_the_builtin_scratch(B):
    """Host-side check, no device needed: n above OG_SORT_NOALLOC_MAX_N is refused before anything is enqueued, and
    the message tells the caller what the limit is and which call to use instead."""
    buf = (C.c_uint64 * 4)()
    in_alt = C.c_int(-1)
    rc = B._lib.og_radix_sort_pairs_noalloc(buf, buf, buf, buf, B.OG_SORT_NOALLOC_MAX_N + 1, 0, 64, C.byref(in_alt), None)
    assert rc == B.OG_ERR_INVALID_ARG
    msg = B._lib.og_last_error().decode()
    assert "OG_SORT_NOALLOC_MAX_N" in msg and str(B.OG_SORT_NOALLOC_MAX_N) in msg and "og_radix_sort_pairs" in msg
    assert in_alt.value == -1                            # untouched
    # the other argument rules are those of og_radix_sort_pairs
    assert B._lib.og_radix_sort_pairs_noalloc(None, buf, buf, buf, 4, 0, 64, None, None) == B.OG_ERR_INVALID_ARG
    assert B._lib.og_radix_sort_pairs_noalloc(buf, buf, buf, buf, 0, 0, 64, None, None) == B.OG_ERR_INVALID_ARG
    assert B._lib.og_radix_sort_pairs_noalloc(buf, buf, buf, buf, 4, 8, 8, None, None) == B.OG_ERR_INVALID_ARG
    # the header's constant is the binding's
    import os
    import re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "og.h")).read()
    assert int(re.search(r"#define\s+OG_SORT_NOALLOC_MAX_N\s+(\d+)u", hdr).group(1)) == B.OG_SORT_NOALLOC_MAX_N


def _keys(rng, n, dup):
    k = rng.integers(0, 1 << 63, n, dtype=np.uint64)
    if n > 1 and dup:
        k[rng.random(n) < dup] = k[0]                    # equal keys: the stable order (index tie-break) is part of the result
    return k


@pytest.mark.gpu
def test_noalloc_sort_equals_the_allocating_path_on_two_calls_in_a_row(B, cuda_device):
    """Two calls back to back on one stream, the second smaller than the first and on another bit range, so that it
    runs over status words, tickets and histograms the first call wrote; then the largest size the array holds and a
    few ragged ones.  Each result is compared with og_radix_sort_pairs (caller-supplied scratch) on the same input:
    keys and values must be identical, and the flag that says which buffer pair holds the result must agree."""
    import torch
    rng = np.random.default_rng(20260617)
    cases = [(300_007, 0, 64, 0.3),                       # 147 tiles, 8 passes, many duplicates
             (70_001, 3, 37, 0.0),                        # second call: fewer tiles, 5 passes (result in the alt pair)
             (B.OG_SORT_NOALLOC_MAX_N, 0, 63, 0.1),       # exactly the limit
             (1, 0, 64, 0.0), (2049, 5, 6, 0.0), (4096, 40, 63, 0.5)]
    # all buffers are made before the first call: the call under test is given memory, it never asks for any
    bufs = []
    for n, b, e, dup in cases:
        k = _keys(rng, n, dup)
        kd = torch.from_numpy(k.view(np.int64)).to(cuda_device)
        bufs.append((k, kd, torch.arange(n, dtype=torch.int32, device=cuda_device), torch.empty_like(kd),
                     torch.empty(n, dtype=torch.int32, device=cuda_device)))
    # the documented set-up call: the first call on a device resolves the built-in array's address (and lets the
    # runtime load the library's device code, which is the one moment device memory may be taken on its behalf)
    w = [torch.zeros(64, dtype=torch.int64, device=cuda_device), torch.arange(64, dtype=torch.int32, device=cuda_device),
         torch.zeros(64, dtype=torch.int64, device=cuda_device), torch.zeros(64, dtype=torch.int32, device=cuda_device)]
    B.og_radix_sort_pairs_noalloc(*w)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    got = []
    for (n, b, e, dup), (k, kd, vd, ka, va) in zip(cases, bufs):
        ks, vs = B.og_radix_sort_pairs_noalloc(kd, vd, ka, va, b, e)     # same stream, no synchronisation in between
        got.append((ks, vs, ks is ka))
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "device memory was taken during the no-alloc calls"
    for (n, b, e, dup), (k, *_), (ks, vs, in_alt) in zip(cases, bufs, got):
        assert in_alt == bool(((e - b + 7) // 8) & 1)
        ks_ref, vs_ref = B.og_radix_sort_pairs(torch.from_numpy(k.view(np.int64)).to(cuda_device),
                                               torch.arange(n, dtype=torch.int32, device=cuda_device), b, e)
        torch.cuda.synchronize()
        assert torch.equal(ks, ks_ref), f"keys differ (n={n}, bits [{b}, {e}))"
        assert torch.equal(vs, vs_ref), f"values differ (n={n}, bits [{b}, {e}))"
        # and the existing path's own contract, so that two equal wrong answers cannot pass
        field = (k >> np.uint64(b)) & np.uint64((1 << (e - b)) - 1)
        assert np.array_equal(vs.cpu().numpy().view(np.uint32), np.argsort(field, kind="stable").astype(np.uint32))
