"""Build csrc/liblq.so for sm_100a with nvcc (cross-compiles without a GPU).

Usage: ``python -m paper_1911_07045_b200.build [--force] [--verbose]``.
The library is kept in-tree (git-ignored) so it travels to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "liblq.so")
SOURCES = ["lq_api.cu", "lq_kernels.cu", "lq_sweep.cu", "lq_sweep_rc.cu", "lq_fixup.cu", "lq_descent.cu", "lq_analyze.cu", "lq_slab.cu", "lq_resident.cu"]
HEADERS = ["lq_internal.cuh", "lq_site.cuh", "lq_sweep.cuh", "lq_sweep_dev.cuh", "lq_ctx.cuh", os.path.join("..", "..", "include", "lq.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC",
              "-cudart", "static"]


def lib_path() -> str:
    return LIB


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    flags = list(NVCC_FLAGS)
    if verbose:
        flags += ["-Xptxas", "-v"]
    objs = []
    procs = []
    for s in SOURCES:
        o = os.path.join(CSRC, s[:-3] + ".o")
        objs.append(o)
        procs.append(subprocess.Popen([nvcc] + flags + ["-c", os.path.join(CSRC, s), "-o", o]))
    for p in procs:
        if p.wait() != 0:
            raise RuntimeError("nvcc failed")
    tmp = LIB + ".tmp%d" % os.getpid()
    subprocess.run([nvcc, "-shared", "-cudart", "static", "-Wno-deprecated-gpu-targets", "-o", tmp] + objs, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
