"""In-tree build of libobem.so (csrc/*.cu -> paper_2110_09214_b200/libobem.so) with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(_HERE)
SRC = os.path.join(_HERE, "csrc", "obem.cu")
SRCS = [SRC, os.path.join(_HERE, "csrc", "obem_next.cu"),           # hot path; adjacent steps
        os.path.join(_HERE, "csrc", "obem_map.cu"), os.path.join(_HERE, "csrc", "obem_near.cu"),
        os.path.join(_HERE, "csrc", "obem_nn.cu"), os.path.join(_HERE, "csrc", "obem_geom.cu"),
        os.path.join(_HERE, "csrc", "obem_multi.cu"), os.path.join(_HERE, "csrc", "obem_static.cu")]
DEPS = SRCS + [os.path.join(_HERE, "csrc", "obem_internal.cuh")]
HDR = os.path.join(ROOT, "include", "obem.h")
LIB = os.path.join(_HERE, "libobem.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",  # cudart is linked statically (nvcc default): no search-path dependency
    "--threads", "0",                  # the translation units compile in parallel
]


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: libobem.so cannot be built (there is no CPU fallback)")
    return p


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in DEPS + [HDR])


def build_lib(force: bool = False, verbose: bool = False) -> str:
    """Compile the CUDA library if it is missing or older than its sources.  Returns its path."""
    if not force and not is_stale():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [
        "-I", os.path.join(ROOT, "include"), "-o", tmp] + SRCS
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_lib(force=True, verbose=True))
