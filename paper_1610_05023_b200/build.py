"""Builds the C-ABI shared library `libdg_habc.so` in-tree with nvcc for sm_100a (no torch involved)."""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdg_habc.so")
SOURCES = ["dg_api.cu", "mesh.cpp", "refelem.cpp"]
HEADERS = ["kernels.cuh", "kernels_aux.cuh", "kernel_face2d.cuh", "kernel_vol3d_mma.cuh", "kernel_vol3d_ws.cuh", "kernel_vol3d_tf32.cuh", "kernel_vol3d_mmag.cuh", "kernel_vol3d_tf32g.cuh", "kernel_vol3d_elem.cuh", "mesh.hpp", "refelem.hpp", "habc_coef.hpp",
           os.path.join("..", "..", "include", "dg_habc.h")]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA toolkit is required to build libdg_habc.so")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/ into libdg_habc.so (sm_100a, -lineinfo).  Returns the library path."""
    if not force and not is_stale():
        return LIB
    cmd = [_nvcc(), "-O3", "-std=c++17", "-shared", "-Xcompiler", "-fPIC",
           "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
