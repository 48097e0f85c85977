"""Build paper_2303_12166_b200/libnb.so (C ABI of include/nb.h) with nvcc for sm_100a.

In-tree, explicit nvcc: the .so travels to the GPU box with the repo snapshot.
nvcc cross-compiles without a GPU.  Run as `python -m paper_2303_12166_b200.build`.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libnb.so")
SOURCES = [os.path.join(CSRC, "nb_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "nb_kernels.cuh"), os.path.join(CSRC, "nb_cells.cuh"), os.path.join(CSRC, "nb_fused.cuh"),
                  os.path.join(ROOT, "include", "nb.h")]

NVCC_FLAGS = [
    "-std=c++17", "-O3", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "--shared", "-Xcompiler", "-fPIC",
    "-I", os.path.join(ROOT, "include"), "-I", CSRC,
]


def build(force: bool = False, verbose: bool = False) -> str:
    lib = LIB
    if not force and os.path.exists(lib) and all(
            os.path.getmtime(lib) >= os.path.getmtime(d) for d in DEPS):
        return lib
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + SOURCES
    subprocess.check_call(cmd)
    return lib


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv))
