"""Build paper_2001_02765_b200/libsg_disk.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsg_disk.so")
SOURCES = ["sg_layout.cpp", "sg_kernels.cu", "sg_kernels_lin.cu", "sg_kernels_patch.cu", "sg_kernels_lattice.cu", "sg_api.cu", "sg_static.cu"]
HEADERS = ["sg_layout.h", "sg_kernels.cuh", "sg_device.cuh", "sg_kernels_lin.cuh", "sg_kernels_patch.cuh", "sg_patch_device.cuh", "sg_kernels_lattice.cuh", os.path.join("..", "..", "include", "sg_disk.h"), os.path.join("..", "..", "include", "sg_disk_diag.h"), os.path.join("..", "..", "include", "sg_disk_static.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-Xcompiler", "-O3", "-Xcompiler", "-fopenmp", "--shared", "-cudart", "shared", "-lgomp"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []),
           "-o", LIB, *[os.path.join(CSRC, f) for f in SOURCES]]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
