"""Builds the C-ABI library libdd_b200.so (CUDA, sm_100a) in-tree with nvcc.

    python -m paper_1201_5380_b200.build [--force]

nvcc cross-compiles without a GPU.  Every source is compiled to an object file of its own (in parallel, only when
it or a header changed) under build/ at the repo root, then linked.  The built .so is git-ignored but travels to
the GPU box with the gpurun snapshot; the ptxas report (registers, spills) of the last build of every source is
kept beside its object file as build/obj/<source>.ptxas.log.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libdd_b200.so")
OBJ = os.path.join(os.path.dirname(_HERE), "build", "obj")
SOURCES = ["dd_api.cu", "dd_kernels.cu", "dd_kernel_v1.cu", "dd_kernel_v2.cu", "dd_kernel_bp.cu", "dd_kernel_gs.cu", "dd_kernel_gr.cu",
           "dd_scrunch.cu", "dd_scrunch_set.cu", "dd_tree.cu", "dd_plan.cpp"]
HEADERS = ["dd_plan.h", "dd_kernels.cuh", "dd_common.cuh", "dd_bp_core.cuh", os.path.join("..", "..", "include", "dd.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xptxas", "-v",
]


def _mtime(path: str) -> float:
    return os.path.getmtime(path) if os.path.exists(path) else 0.0


def _compile(nvcc: str, src: str, verbose: bool) -> str:
    obj = os.path.join(OBJ, src + ".o")
    r = subprocess.run([nvcc, *NVCC_FLAGS, "-c", "-o", obj, os.path.join(CSRC, src)], capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed on {src}")
    with open(os.path.join(OBJ, src + ".ptxas.log"), "w") as f:
        f.write(r.stdout + r.stderr)
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    newest_header = max([_mtime(os.path.join(CSRC, h)) for h in HEADERS] + [_mtime(os.path.abspath(__file__))])
    stale = [s for s in SOURCES
             if force or _mtime(os.path.join(OBJ, s + ".o")) < max(_mtime(os.path.join(CSRC, s)), newest_header)]
    if not stale and _mtime(LIB) >= max(_mtime(os.path.join(OBJ, s + ".o")) for s in SOURCES):
        return LIB
    with ThreadPoolExecutor(max_workers=min(len(stale), os.cpu_count() or 1) or 1) as pool:
        list(pool.map(lambda s: _compile(nvcc, s, verbose), stale))
    cmd = [nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB + ".tmp"] + \
          [os.path.join(OBJ, s + ".o") for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed linking libdd_b200.so")
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
