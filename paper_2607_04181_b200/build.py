"""Builds libcocoscale.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2607_04181_b200.build [--force] [-v] [--trace]

--trace builds libcocoscale_trace.so, the same sources with -DCC_TRACE (globaltimer trace points, timeline.py).

nvcc cross-compiles without a GPU.  The library lands next to this file so that it travels with
the repository snapshot to the GPU box; it is git-ignored.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcocoscale.so")
SOURCES = ["cc_api.cu", "cc_kernels.cu", "cc_rowwise.cu", "cc_gemm.cu", "cc_attention.cu", "cc_control.cu", "cc_big.cu", "cc_big_gemm.cu",
           "cc_prefill.cu", "cc_noalloc.cu"]
HEADERS = ["cc_common.cuh", "cc_kernels.h", "cc_epilogue.cuh", os.path.join("..", "..", "include", "cocoscale.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-fvisibility=hidden", "--threads", "4"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


LIB_TRACE = os.path.join(HERE, "libcocoscale_trace.so")   # the same sources with -DCC_TRACE (timeline.py)


def needs_build(trace: bool = False) -> bool:
    lib = LIB_TRACE if trace else LIB
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> str:
    lib = LIB_TRACE if trace else LIB
    if not force and not needs_build(trace):
        return lib
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src.replace(".cu", ".trace.o" if trace else ".o"))
        cmd = [_nvcc(), *NVCC_FLAGS, *(["-DCC_TRACE"] if trace else []), "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if verbose and out:
            print(out)
        if p.returncode:
            raise RuntimeError(f"nvcc failed on {src}:\n{out}")
    tmp = lib + ".tmp"
    link = [_nvcc(), "-shared", "-o", tmp, *objs, "-cudart", "static", "-Xlinker", "--no-undefined", "-lpthread", "-ldl", "-lrt"]
    r = subprocess.run(link, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if r.returncode:
        raise RuntimeError("link failed:\n" + r.stdout)
    os.replace(tmp, lib)
    for o in objs:
        os.remove(o)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv))
