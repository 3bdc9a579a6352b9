"""Builds libogtree.so (hand-written CUDA for sm_100a; the product) and libogprobe.so (the FP32 throughput
probe bench.py uses to state the measured ALU rate; not part of the product ABI) in-tree with nvcc.

    python -m paper_2606_17145_b200.build [--force]

nvcc cross-compiles without a GPU.  The library is kept beside the package so that it travels
with the tree to the GPU box; it is git-ignored (source-only history).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libogtree.so")
PROBE_LIB = os.path.join(HERE, "libogprobe.so")
SOURCES = ["api.cu", "keys.cu", "radix_sort.cu", "octree.cu", "walk.cu", "pm.cu", "timestep.cu", "sph.cu", "let.cu"]
PROBE_SOURCES = ["probe.cu"]
HEADERS = ["og_internal.cuh", "walk_math.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(PROBE_LIB):
        return True
    t = min(os.path.getmtime(LIB), os.path.getmtime(PROBE_LIB))
    deps = [os.path.join(CSRC, s) for s in SOURCES + PROBE_SOURCES + HEADERS] + [os.path.join(ROOT, "include", "og.h"),
                                                                  os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    objs = []
    procs = []
    for s in SOURCES + PROBE_SOURCES:
        o = os.path.join(objdir, s.replace(".cu", ".o"))
        cmd = [_nvcc(), *NVCC_FLAGS, *os.environ.get("OG_NVCC_EXTRA", "").split(), "-I", os.path.join(ROOT, "include"), "-I", CSRC, "-c",
               os.path.join(CSRC, s), "-o", o]
        procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(o)
    log = []
    failed = False
    for s, p in procs:
        out, _ = p.communicate()
        log.append(f"==== {s}\n{out}")
        failed |= p.returncode != 0
    with open(os.path.join(objdir, "ptxas.log"), "w") as f:
        f.write("\n".join(log))
    if failed or verbose:
        sys.stderr.write("\n".join(log))
    if failed:
        raise RuntimeError("nvcc failed (see output above)")
    n = len(SOURCES)
    # static cudart (nvcc default); cuFFT (the DFT of the PM step) from the toolkit's shared library
    subprocess.run([_nvcc(), "-shared", "-o", LIB, *objs[:n], "-lcufft", "-Xlinker", "-rpath=/usr/local/cuda/lib64"],
                   check=True)
    subprocess.run([_nvcc(), "-shared", "-o", PROBE_LIB, *objs[n:]], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
