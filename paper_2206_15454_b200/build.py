"""Build step of the CUDA library: nvcc -> paper_2206_15454_b200/liblbm_b200.so (sm_100a only).

The shared object is built in-tree (git-ignored) so that it travels to the GPU box with the
repository snapshot.  `python -m paper_2206_15454_b200.build [--force] [--verbose]`.

The step kernel exists in ~130 variants (cells per thread x storage mode x statistics x geometry x
SGS table, plus the TMA tiles); they are spread over 15 translation units (csrc/lbm_step_inst.cu and
csrc/lbm_tma_inst.cu compiled once per template-argument set) that compile in parallel, then one link.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(_HERE, "build")
DEPS = [os.path.join(CSRC, f) for f in ("lbm_api.cu", "lbm_static.cu", "lbm_step_inst.cu", "lbm_tma_inst.cu", "lbm_kernels.cuh",
                                         "lbm_tma.cuh", "lbm_launch.cuh")] + [os.path.join(ROOT, "include", "lbm.h")]
LIB = os.path.join(_HERE, "liblbm_b200.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
    # FMA contraction on.  No -use_fast_math: the kernels choose their approximations themselves -
    # MUFU rcp.approx / sqrt.approx with FTZ (inline PTX in lbm_kernels.cuh) for 1/rho, |u|, the two
    # square roots of Eqs. 11-12 and 1/tau, where the error is second order (DESIGN.md "Arithmetic
    # form"); everything else is IEEE fp32.
    "--fmad=true",
    "-Xptxas", "-warn-spills", "-diag-suppress", "177",
]


def units():
    """(object name, source, extra defines) of every translation unit."""
    out = [("lbm_api.o", "lbm_api.cu", []), ("lbm_static.o", "lbm_static.cu", [])]
    for v in (4, 2, 1):
        for s in (0, 1):
            for g in (0, 1):
                out.append((f"lbm_step_v{v}_s{s}_g{g}.o", "lbm_step_inst.cu", [f"-DLBM_V={v}", f"-DLBM_S={s}", f"-DLBM_G={g}"]))
    for s in (0, 1):
        out.append((f"lbm_tma_s{s}.o", "lbm_tma_inst.cu", [f"-DLBM_S={s}"]))
    return out


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: the CUDA library cannot be built")
    return p


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS + [os.path.abspath(__file__)])


def _stale(obj: str, src: str) -> bool:
    """An object is rebuilt when its source, a header it includes or this script is newer."""
    o = os.path.join(OBJ, obj)
    if not os.path.exists(o):
        return True
    deps = [os.path.join(CSRC, src), os.path.join(CSRC, "lbm_kernels.cuh"), os.path.join(CSRC, "lbm_launch.cuh"),
            os.path.abspath(__file__)]
    if src == "lbm_tma_inst.cu":
        deps.append(os.path.join(CSRC, "lbm_tma.cuh"))
    if src in ("lbm_api.cu", "lbm_static.cu"):
        deps.append(os.path.join(ROOT, "include", "lbm.h"))
    t = os.path.getmtime(o)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or needs_build()):
        return LIB
    os.makedirs(OBJ, exist_ok=True)
    nvcc = nvcc_path()
    todo = [u for u in units() if force or _stale(u[0], u[1])]

    def compile_one(u):
        obj, src, defs = u
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + defs + [
            "-c", os.path.join(CSRC, src), "-o", os.path.join(OBJ, obj)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        return obj, cmd, r

    jobs = max(1, min(len(todo), os.cpu_count() or 1))
    with ThreadPoolExecutor(jobs) as ex:
        results = list(ex.map(compile_one, todo))
    for obj, cmd, r in results:
        if verbose:
            print(" ".join(cmd), file=sys.stderr)
        if r.stderr.strip() and (verbose or r.returncode != 0):
            print(r.stderr, file=sys.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {obj}")
    link = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", LIB] + [
        os.path.join(OBJ, u[0]) for u in units()]
    if verbose:
        print(" ".join(link), file=sys.stderr)
    subprocess.check_call(link)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
