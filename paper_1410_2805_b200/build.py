"""Compile csrc/*.cu into paper_1410_2805_b200/libhaccsr.so for sm_100a (nvcc, in-tree).

`python -m paper_1410_2805_b200.build` rebuilds; `build()` is what __graft_entry__.build()
and the Python binding call.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import glob
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhaccsr.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
    "--fmad=false",  # every FMA in the kernels is written explicitly
    "-Xptxas", "-v",
]


def _sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return _sources() + glob.glob(os.path.join(CSRC, "*.h")) + \
        glob.glob(os.path.join(INCLUDE, "*.h")) + [os.path.abspath(__file__)]


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    return all(os.path.getmtime(p) <= t for p in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and up_to_date():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, *NVCC_FLAGS, "-I", INCLUDE, "-o", LIB, *_sources()]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        print(r.stdout)
        print(r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libhaccsr.so")
    return LIB


# ---- libhaccpm.so: the long-range PM force (csrc_pm/, links cuFFT) -----------------------
CSRC_PM = os.path.join(HERE, "csrc_pm")
LIB_PM = os.path.join(HERE, "libhaccpm.so")


def _pm_deps():
    return sorted(glob.glob(os.path.join(CSRC_PM, "*.cu"))) + \
        [os.path.join(INCLUDE, "haccpm.h"), os.path.abspath(__file__)]


def build_pm(force: bool = False, verbose: bool = False) -> str:
    if (not force and os.path.exists(LIB_PM)
            and all(os.path.getmtime(p) <= os.path.getmtime(LIB_PM) for p in _pm_deps())):
        return LIB_PM
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, *NVCC_FLAGS, "-I", INCLUDE, "-o", LIB_PM,
           *sorted(glob.glob(os.path.join(CSRC_PM, "*.cu"))), "-lcufft"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        print(r.stdout)
        print(r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libhaccpm.so")
    return LIB_PM


if __name__ == "__main__":
    print(build_pm(force=True, verbose=True))
    print(build(force=True, verbose=True))
