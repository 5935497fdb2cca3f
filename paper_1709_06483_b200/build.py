"""Build libmagnus_b200.so in-tree with nvcc for sm_100a.  `python -m paper_1709_06483_b200.build`.

The shared library is the product's C-ABI boundary (include/magnus.h); the
Python binding only marshals arguments into it.  nvcc cross-compiles without a
GPU, so this also runs on the CPU-only build box.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmagnus_b200.so")

CU_SOURCES = ["api.cu", "kernels_common.cu", "kernels_csr.cu", "kernels_csr_rowblock.cu", "kernels_csr_small.cu", "kernels_csr_mid.cu", "kernels_csr_slice.cu", "kernels_csr_stream.cu", "kernels_dense.cu", "kernels_dense_sweep.cu", "kernels_xxz.cu", "kernels_lanczos.cu",
              "zgemm_dmma.cu", "no_alloc.cu"]
CPP_SOURCES = ["host_leja.cpp"]
HEADERS = ["magnus_internal.h", "device_utils.cuh", "leja_finalize.cuh", os.path.join("..", "..", "include", "magnus.h")]

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-Xptxas", "-v", *ARCH]
CXX_FLAGS = ["-O2", "-std=c++17", "-fPIC", "-Wall", "-Wextra"]


def _newer(src: str, dst: str) -> bool:
    return (not os.path.exists(dst)) or os.path.getmtime(src) > os.path.getmtime(dst)


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(BUILD, exist_ok=True)
    header_paths = [os.path.join(CSRC, h) for h in HEADERS]
    objs = []
    relink = force or not os.path.exists(LIB)
    for name in CU_SOURCES + CPP_SOURCES:
        src = os.path.join(CSRC, name)
        obj = os.path.join(BUILD, name + ".o")
        objs.append(obj)
        stale = force or _newer(src, obj) or any(_newer(h, obj) for h in header_paths)
        if not stale:
            continue
        relink = True
        if name.endswith(".cu"):
            cmd = [NVCC, *NVCC_FLAGS, "-c", src, "-o", obj]
        else:
            cmd = ["g++", *CXX_FLAGS, "-c", src, "-o", obj]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError(f"compilation of {name} failed")
        with open(obj + ".log", "w") as fh:          # ptxas -v output: registers, spills, shared memory
            fh.write(res.stdout + res.stderr)
    if relink:
        cmd = [NVCC, "-shared", *ARCH, "-o", LIB, *objs]
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            sys.stderr.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
            raise RuntimeError("link failed")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
