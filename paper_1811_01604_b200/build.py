"""In-tree build of the CUDA library (sm_100a only).

`python -m paper_1811_01604_b200.build` or `build()` compiles csrc/*.cu into
paper_1811_01604_b200/libmpr_b200.so with nvcc (cross-compiles without a GPU).
"""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libmpr_b200.so")
SOURCES = ["mpr_api.cu"]
HEADERS = ["mpr_device.cuh", "mpr_f64.cuh", "mpr_f64_api.inl", "mpr_noalloc.inl"]
# pipe-rate micro-benchmarks behind `bench.py --sfu-peak` (the roofline's measured denominators); not part of the MPR library
MICROBENCH_LIB = os.path.join(_HERE, "libmpr_microbench.so")
MICROBENCH_SOURCES = ["mpr_microbench.cu"]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "--cudart", "static",
]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(INCLUDE, "mpr.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build_microbench(force: bool = False) -> str:
    srcs = [os.path.join(CSRC, f) for f in MICROBENCH_SOURCES]
    if force or not os.path.exists(MICROBENCH_LIB) or any(os.path.getmtime(f) > os.path.getmtime(MICROBENCH_LIB) for f in srcs):
        subprocess.run([_nvcc(), *NVCC_FLAGS, "-o", MICROBENCH_LIB] + srcs, check=True)
    return MICROBENCH_LIB


CHECKED_LIB = os.path.join(_HERE, "libmpr_b200_checked.so")


def build_checked(force: bool = False) -> str:
    """The library with -DMPR_CHECKED: device-side assertions on every shared-memory and accumulator index of the tile
    passes (a stand-in for compute-sanitizer memcheck where that is not available).  `tests/sanitizer_driver.py --lib`."""
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS]
    if force or not os.path.exists(CHECKED_LIB) or any(os.path.getmtime(d) > os.path.getmtime(CHECKED_LIB) for d in deps):
        subprocess.run([_nvcc(), *NVCC_FLAGS, "-DMPR_CHECKED", "-I", INCLUDE, "-o", CHECKED_LIB] +
                       [os.path.join(CSRC, f) for f in SOURCES], check=True)
    return CHECKED_LIB


def build(force: bool = False, verbose: bool = False) -> str:
    build_microbench(force)
    if force or _stale():
        cmd = [_nvcc(), *NVCC_FLAGS, "-I", INCLUDE, "-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
        if verbose:
            cmd.insert(1, "-Xptxas")
            cmd.insert(2, "-v")
            print(" ".join(cmd))
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
