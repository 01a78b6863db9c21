"""Build libkspw.so (hand-written CUDA for sm_100a) in-tree with nvcc.  No torch extension machinery:
the library is a plain C-ABI shared object (include/kspw.h) loaded with ctypes."""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libkspw.so")
SOURCES = ["capi.cu", "hpsi_kernels.cu", "gemm.cu", "eigh.cu", "davidson.cu", "cg.cu", "batch.cu"]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-Wno-deprecated-gpu-targets"]


FLAGS += os.environ.get("KSPW_NVCC_FLAGS", "").split()      # e.g. -DKSPW_NO_YHALF (compile-time switches of DESIGN.md §9)


def _newest_header() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, f)) for f in os.listdir(CSRC) if f.endswith((".h", ".cuh")))


def _compile(src: str, force: bool) -> str:
    obj = os.path.join(OBJ, src.replace(".cu", ".o"))
    s = os.path.join(CSRC, src)
    if (not force and os.path.exists(obj)
            and os.path.getmtime(obj) >= max(os.path.getmtime(s), _newest_header())):
        return obj
    subprocess.check_call([NVCC] + FLAGS + ["-c", s, "-o", obj])
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    with cf.ThreadPoolExecutor(max_workers=min(len(SOURCES), os.cpu_count() or 1)) as ex:
        objs = list(ex.map(lambda s: _compile(s, force), SOURCES))
    if force or not os.path.exists(LIB) or any(os.path.getmtime(o) > os.path.getmtime(LIB) for o in objs):
        tmp = LIB + ".tmp%d" % os.getpid()
        subprocess.check_call([NVCC, "-shared", "-Wno-deprecated-gpu-targets", "-o", tmp] + objs + ["-lcudart"])
        os.replace(tmp, LIB)
        if verbose:
            print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
