"""Builds the CUDA extension in-tree: paper_1912_09161_b200/_allen_velo.so (sm_100a, -lineinfo).

nvcc cross-compiles without a GPU.  The shared object has a plain C ABI (include/allen_velo.h) and links the CUDA
runtime statically; it does not depend on torch.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "_allen_velo.so")
LIB_DEBUG = os.path.join(HERE, "_allen_velo_debug.so")  # the same sources with -DVELO_DEBUG (bounds checks)
SOURCES = ["allen_velo.cu", "velo_cluster.cu", "velo_scan.cu", "velo_track.cu", "velo_seed.cu", "velo_follow.cu", "velo_pv.cu"]
# include/allen_velo_noalloc.h: its own translation unit (static device scratch array), outside csrc/
SOURCES.append(os.path.join("..", "csrc_noalloc", "offsets_static.cu"))
HEADERS = ["velo_common.cuh", "velo_track.cuh", os.path.join("..", "..", "include", "allen_velo.h"),
           os.path.join("..", "..", "include", "allen_velo_debug.h"),
           os.path.join("..", "..", "include", "allen_velo_noalloc.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-fmad=false",
]


def _stale(lib=LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, debug: bool = False) -> str:
    lib = LIB_DEBUG if debug else LIB
    if not force and not _stale(lib):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = lib + f".{os.getpid()}.tmp"
    cmd = ([nvcc] + NVCC_FLAGS + (["-DVELO_DEBUG"] if debug else []) + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp]
           + [os.path.join(CSRC, s) for s in SOURCES])
    subprocess.check_call(cmd)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, debug="--debug" in sys.argv))
