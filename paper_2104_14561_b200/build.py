"""Build the CUDA path in-tree: csrc/*.cu -> paper_2104_14561_b200/libfk_b200.so (sm_100a only).

`python -m paper_2104_14561_b200.build` or `build_library()`; nvcc cross-compiles without a
GPU.  The library is rebuilt when a source or header is newer than it.
"""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
LIB_PATH = os.path.join(_HERE, "libfk_b200.so")
SOURCES = [os.path.join(_HERE, "csrc", f) for f in ("fk_api.cu", "fk_kernels.cu", "fk_fused2d.cu", "fk_rowblock3d.cu", "fk_far2d.cu", "fk_line1d.cu", "fk_peak.cu")]
HEADERS = [os.path.join(_HERE, "csrc", "fk_internal.h"), os.path.join(_HERE, "csrc", "fk_device.cuh"), os.path.join(_ROOT, "include", "fk.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: cannot build libfk_b200.so")


def stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS)


def build_library(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB_PATH] + SOURCES
        res = subprocess.run(cmd, capture_output=True, text=True)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
        if verbose:
            print(res.stderr)
    return LIB_PATH


if __name__ == "__main__":
    print(build_library(force=True, verbose=True))
