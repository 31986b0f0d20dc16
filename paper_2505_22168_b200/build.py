"""Builds libgmnn_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2505_22168_b200.build [--force] [--verbose]

The shared object is git-ignored but travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
# GMNN_B200_LIB: build to / load from another path (e.g. a -DGMNN_EXPERIMENTS build kept beside the shipped one)
LIB = os.environ.get("GMNN_B200_LIB") or os.path.join(HERE, "libgmnn_b200.so")
SOURCES = ["gmnn_api.cu", "neighbor.cu", "descriptor.cu", "pair_forward.cu", "pair_backward.cu", "mlp_simt.cu", "mlp_tc.cu", "md.cu"]
HEADERS = ["gmnn_internal.h", "contraction.cuh", "pair_common.cuh", "tc_ptx.cuh", os.path.join("..", "..", "include", "gmnn.h")]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-cudart", "static", "--expt-relaxed-constexpr",
]


if os.environ.get("GMNN_EXPERIMENTS"):  # knock-out / superseded-variant knobs for timing studies (never shipped)
    NVCC_FLAGS.append("-DGMNN_EXPERIMENTS")


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    objdir = os.path.join(HERE, "build_experiments" if os.environ.get("GMNN_EXPERIMENTS") else "build")
    os.makedirs(objdir, exist_ok=True)
    hdrs = [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS]
    objs = []
    procs = []
    for src in SOURCES:
        sp = os.path.join(CSRC, src)
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        objs.append(obj)
        if force or _stale(obj, [sp, *hdrs]):
            cmd = [_nvcc(), *NVCC_FLAGS, "-c", sp, "-o", obj]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
                print(" ".join(cmd), flush=True)
            procs.append((src, subprocess.Popen(cmd)))
    failed = [src for src, p in procs if p.wait() != 0]
    if failed:
        raise RuntimeError("nvcc failed for: " + ", ".join(failed))
    if force or procs or _stale(LIB, objs):
        cmd = [_nvcc(), "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", *objs, "-o", LIB]
        if verbose:
            print(" ".join(cmd), flush=True)
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
