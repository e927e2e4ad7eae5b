"""Build libdbie_b200.so (CUDA, sm_100a) and the host test shim, in-tree.

    python -m paper_1306_1122_b200.build [--force] [-v]

nvcc cross-compiles without a GPU.  The shared objects are git-ignored but travel to the GPU
box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libdbie_b200.so")
SHIM = os.path.join(HERE, "libdbie_hostshim.so")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", INCLUDE]

# (source, extra flags).  dbie_solver.cu is compiled without FMA contraction: the simplex
# decisions are comparisons of separately rounded IEEE operations.
UNITS = [
    ("dbie_interact.cu", []),
    ("dbie_solve_fused.cu", []),     # same flags as dbie_interact.cu: identical interaction arithmetic
    ("dbie_solver.cu", ["-fmad=false"]),
    ("dbie_grid.cu", ["-fmad=false"]),
    ("dbie_trace.cu", ["-fmad=false"]),
    ("dbie_api.cu", []),
]
HEADERS = ["dbie_internal.h", "dbie_interact_fp64.cuh", "dbie_tma.cuh", "dbie_math.cuh", "dbie_math_f32.cuh", "dbie_nm.cuh", "dbie_solver_common.cuh",
           "trig_coeffs.h", "trig_coeffs_f32.h"]


def _newer(target: str, deps: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build_lib(force: bool = False, verbose: bool = False) -> str:
    deps = [os.path.join(CSRC, h) for h in HEADERS] + [os.path.join(INCLUDE, "dbie.h"),
                                                     os.path.abspath(__file__)]
    objs = []
    for src, extra in UNITS:
        s = os.path.join(CSRC, src)
        o = os.path.join(CSRC, src.replace(".cu", ".o"))
        if force or _newer(o, deps + [s]):
            cmd = [NVCC, *ARCH, *COMMON, *extra, "-c", s, "-o", o]
            if verbose:
                cmd.insert(1, "-Xptxas=-v")
            subprocess.check_call(cmd)
        objs.append(o)
    if force or _newer(LIB, objs):
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call([NVCC, *ARCH, "-shared", "-o", tmp, *objs])
        os.replace(tmp, LIB)
    return LIB


def build_hostshim(force: bool = False) -> str:
    """CPU build of the __host__ __device__ arithmetic headers, for the not-gpu tests."""
    src = os.path.join(CSRC, "host_shim.cpp")
    deps = [src] + [os.path.join(CSRC, h) for h in ("dbie_math.cuh", "dbie_math_f32.cuh", "dbie_nm.cuh", "trig_coeffs.h",
                                                     "trig_coeffs_f32.h")]
    if force or _newer(SHIM, deps):
        tmp = SHIM + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math",
                               "-shared", "-fPIC", "-x", "c++", src, "-o", tmp, "-lm"])
        os.replace(tmp, SHIM)
    return SHIM


def build_all(force: bool = False, verbose: bool = False) -> None:
    build_lib(force, verbose)
    build_hostshim(force)


if __name__ == "__main__":
    build_all(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print(LIB)
    print(SHIM)
