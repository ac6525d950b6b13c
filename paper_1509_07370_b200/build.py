"""Builds libbh.so in-tree with nvcc for sm_100a (B200).  `python -m paper_1509_07370_b200.build`."""
from __future__ import annotations

import glob
import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libbh.so")
CHECKED_LIB = os.path.join(HERE, "libbh_checked.so")   # -DBH_CHECKED: device-side bounds checks (tests/test_gpu_checked.py)
PEAK_LIB = os.path.join(HERE, "libbh_fma_peak.so")      # bench.py's measured FP32 denominator; not part of libbh
PEAK_SRC = os.path.join(CSRC, "fma_peak.cu")
LIB_SRCS = [os.path.join(CSRC, "bh.cu"), os.path.join(CSRC, "direct_noalloc.cu")]   # the translation units of libbh
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libbh needs the CUDA toolkit (there is no CPU fallback)")


def sources():
    return sorted([s for s in glob.glob(os.path.join(CSRC, "*.cu")) if s != PEAK_SRC] +
                  glob.glob(os.path.join(CSRC, "*.cuh")) + [os.path.join(os.path.dirname(HERE), "include", "bh.h")])


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in sources())


def build(force: bool = False, verbose: bool = False) -> str:
    """nvcc -gencode arch=compute_100a,code=sm_100a ... -> paper_1509_07370_b200/libbh.so"""
    if force or needs_build():
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + LIB_SRCS
        subprocess.check_call(cmd)
    return LIB


def build_checked(force: bool = False) -> str:
    """The same library with -DBH_CHECKED: every index the kernels compute is bounds-checked on the device."""
    if force or not os.path.exists(CHECKED_LIB) or any(os.path.getmtime(s) > os.path.getmtime(CHECKED_LIB) for s in sources()):
        subprocess.check_call([_nvcc()] + NVCC_FLAGS + ["-DBH_CHECKED", "-o", CHECKED_LIB] + LIB_SRCS)
    return CHECKED_LIB


def build_fma_peak(force: bool = False) -> str:
    """The FMA-chain peak measurement bench.py reports beside the nominal FP32 peak (its own small library)."""
    if force or not os.path.exists(PEAK_LIB) or os.path.getmtime(PEAK_LIB) < os.path.getmtime(PEAK_SRC):
        subprocess.check_call([_nvcc()] + NVCC_FLAGS + ["-o", PEAK_LIB, PEAK_SRC])
    return PEAK_LIB


if os.environ.get("BH_CHECKED") == "1":       # debugging aid: the binding loads the checked build instead
    LIB = CHECKED_LIB
    build = build_checked                         # noqa: F811


if __name__ == "__main__":
    if "--checked" in sys.argv:
        print(build_checked(force="--force" in sys.argv))
    else:
        print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
        print(build_fma_peak(force="--force" in sys.argv))
