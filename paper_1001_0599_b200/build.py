"""Build libcbct.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1001_0599_b200.build [--force]

nvcc cross-compiles without a GPU.  The shared object lands next to this file so that it
travels with the repository snapshot to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libcbct.so")
SOURCES = ["geometry.cu", "forward.cu", "back.cu", "back_tma.cu", "back_eq6.cu", "tv.cu", "transfer.cu", "metrics.cu", "metrics_static.cu", "fbs.cu", "calib.cu"]
HEADERS = ["cbct_internal.cuh", "ray.cuh", "reduce.cuh", os.path.join("..", "..", "include", "cbct.h")]
# static cudart (nvcc's default): no run-time dependency on a libcudart path; device pointers and
# streams made by torch's runtime are valid here because both use the device's primary context.
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-O2", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or stale()):
        return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + os.environ.get("CBCT_NVCC_EXTRA", "").split()
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
