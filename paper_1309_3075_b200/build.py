"""Build libepx.so (the C-ABI library of include/epx.h) in-tree with nvcc for sm_100a.

``python -m paper_1309_3075_b200.build`` or ``build_library()``.  nvcc cross-compiles without a GPU.  The .so sits
next to this file so that it travels to the GPU box with the repo snapshot (it is git-ignored).
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libepx.so")
SOURCES = ["api.cu", "segmenter.cu", "eigen.cu", "chain.cu", "pade.cu", "prune.cu", "prune_lane.cu", "prune_mma.cu", "peaks.cu"]
DEPS = ["epx_internal.h", "prune_common.cuh", "seg_common.cuh", "api_compute.inc", os.path.join("..", "..", "include", "epx.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"] + os.environ.get("EPX_NVCC_EXTRA", "").split()


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libepx.so cannot be built (there is no CPU fallback)")
    return exe


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build_library(force: bool = False, verbose: bool = False) -> str:
    nvcc = _nvcc()
    objdir = os.path.join(_HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    common = [os.path.join(CSRC, d) for d in DEPS] + [os.path.abspath(__file__)]
    objs, procs = [], []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(objdir, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + common):
            cmd = [nvcc] + NVCC_FLAGS + ["-c", s, "-o", o]
            if verbose:
                cmd[1:1] = ["-Xptxas", "-v"]
            procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write(f"--- nvcc {src}\n{out}\n")
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    if procs or force or _stale(LIB_PATH, objs):
        # static cudart (nvcc default): the library shares the primary context with the caller (torch), so device
        # pointers and cudaStream_t handles are interchangeable
        subprocess.run([nvcc, "-shared", "-o", LIB_PATH] + objs, check=True)
    return LIB_PATH


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
