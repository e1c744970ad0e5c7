"""Build the CUDA library in-tree for sm_100a:  python -m paper_1609_08621_b200.build [--force]

nvcc cross-compiles without a GPU; the resulting libpkdg.so sits next to this file (git-ignored,
but it travels to the GPU box with the working tree).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = os.path.join(HERE, "csrc", "pkdg.cu")
DEPS = [SRC, os.path.join(HERE, "csrc", "pkdg_kernels.cuh"), os.path.join(HERE, "csrc", "pkdg_fmm.cuh"),
        os.path.join(HERE, "csrc", "pkdg_fmm_gen.cuh"), os.path.join(ROOT, "include", "pkdg.h")]
LIB = os.path.join(HERE, "libpkdg.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-shared"]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp, SRC]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
