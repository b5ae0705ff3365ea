"""Build step of the CUDA extension: nvcc -> paper_2511_03683_b200/libephc.so (in-tree, sm_100a only)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libephc.so")
SOURCES = ("ephc_build.cpp", "ephc_tiles.cpp", "ephc_rows.cpp", "ephc_stream.cpp", "ephc_res.cpp", "ephc_api.cu")
HEADERS = ("ephc_internal.h", "ephc_select_kernels.cuh", "ephc_kernels.cuh", "ephc_tile_kernels.cuh", "ephc_row_kernels.cuh", "ephc_stream_kernels.cuh", "ephc_res_kernels.cuh", "ephc_paper_kernels.cuh", os.path.join("..", "..", "include", "ephc.h"))


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def nvcc_path() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if c and os.path.exists(c):
            return c
    return "nvcc"


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the library if it is missing or older than its sources.  Returns the path of the .so."""
    if not force and not _stale():
        return LIB
    tmp = LIB + f".{os.getpid()}.tmp"
    cmd = [nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC,-fopenmp,-O2,-ffp-contract=off", "-shared", "-o", tmp]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += os.environ.get("EPHC_BUILD_FLAGS", "").split()   # e.g. -DEPHC_RES_TIMING for a working build
    cmd += [os.path.join(CSRC, f) for f in SOURCES] + ["-lgomp"]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
