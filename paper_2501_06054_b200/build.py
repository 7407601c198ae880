"""Builds libsas_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libsas_b200.so")
SOURCES = ["sas_api.cu", "reduce_static.cu", "quadrature_host.cpp"]
HEADERS = ["device_math.cuh", "j1_f64_generated.h", "geometry.cuh", "models.cuh", "trace_kernel.cuh", "trace_kernel_ws.cuh", "reduce_kernel.cuh", "sas_types.h",
           "quadrature_host.h", "coeffs_generated.h", os.path.join("..", "..", "include", "sas.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    # the fp64 geometry must keep one rounding per written operation (DESIGN.md R-C0); code that
    # wants fused multiply-adds calls fma()/fmaf() explicitly
    "-fmad=false",
    "-Xcompiler", "-fPIC,-ffp-contract=off", "-shared",
]


def extra_flags() -> list:
    """SAS_DEBUG_BOUNDS=1 in the environment builds the bounds-checking variant (csrc/sas_types.h: SAS_CHECK)."""
    return ["-DSAS_DEBUG_BOUNDS"] if os.environ.get("SAS_DEBUG_BOUNDS", "0") not in ("", "0") else []


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    try:
        if open(LIB + ".flags").read() != " ".join(extra_flags()):
            return True
    except OSError:
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or is_stale():
        cmd = ["nvcc"] + NVCC_FLAGS + extra_flags() + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
        subprocess.check_call(cmd, cwd=CSRC)
        open(LIB + ".flags", "w").write(" ".join(extra_flags()))
    return LIB


def build_microbench() -> str:
    """csrc/microbench.cu -> paper_2501_06054_b200/microbench (pipe rates for the roofline, DESIGN.md s.7)."""
    exe = os.path.join(HERE, "microbench")
    subprocess.check_call(["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17",
                           "-o", exe, "microbench.cu"], cwd=CSRC)
    return exe


if __name__ == "__main__":
    import sys
    if "--microbench" in sys.argv:
        print(build_microbench())
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
