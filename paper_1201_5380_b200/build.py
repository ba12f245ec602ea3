"""Builds the C-ABI library libdd_b200.so (CUDA, sm_100a) in-tree with nvcc.

    python -m paper_1201_5380_b200.build [--force]

nvcc cross-compiles without a GPU.  The built .so is git-ignored but travels to the GPU box with
the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libdd_b200.so")
SOURCES = ["dd_api.cu", "dd_kernels.cu", "dd_kernel_v1.cu", "dd_kernel_v2.cu", "dd_kernel_bp.cu", "dd_scrunch.cu", "dd_scrunch_set.cu", "dd_plan.cpp"]
HEADERS = ["dd_plan.h", "dd_kernels.cuh", "dd_common.cuh", os.path.join("..", "..", "include", "dd.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v",
]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("DD_NVCC_EXTRA", "").split()      # e.g. -DDD_EXPERIMENT=1 for kernel experiments
    cmd = [nvcc, *NVCC_FLAGS, *extra, "-o", LIB + ".tmp"] + [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libdd_b200.so")
    with open(os.path.join(_HERE, "build_ptxas.log"), "w") as f:
        # registers / spills / barriers per kernel; compile times dropped so that the log is reproducible
        f.write("".join(l for l in (r.stdout + r.stderr).splitlines(True) if "Compile time" not in l))
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
