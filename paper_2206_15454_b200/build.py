"""Build step of the CUDA library: nvcc -> paper_2206_15454_b200/liblbm_b200.so (sm_100a only).

The shared object is built in-tree (git-ignored) so that it travels to the GPU box with the
repository snapshot.  `python -m paper_2206_15454_b200.build [--force] [--verbose]`.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(_HERE)
SRC = [os.path.join(_HERE, "csrc", "lbm_api.cu")]
DEPS = SRC + [os.path.join(_HERE, "csrc", "lbm_kernels.cuh"), os.path.join(_HERE, "csrc", "lbm_tma.cuh"),
              os.path.join(ROOT, "include", "lbm.h")]
LIB = os.path.join(_HERE, "liblbm_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    # FMA contraction on.  No -use_fast_math: the kernels choose their approximations themselves -
    # MUFU rcp.approx / sqrt.approx with FTZ (inline PTX in lbm_kernels.cuh) for 1/rho, |u|, the two
    # square roots of Eqs. 11-12 and 1/tau, where the error is second order (DESIGN.md "Arithmetic
    # form"); everything else is IEEE fp32.
    "--fmad=true",
    "-Xptxas", "-warn-spills", "-diag-suppress", "177",
]


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: the CUDA library cannot be built")
    return p


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        cmd = [nvcc_path()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SRC
        if verbose:
            print(" ".join(cmd), file=sys.stderr)
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
