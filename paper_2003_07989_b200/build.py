"""Build the C-ABI shared library `librips_b200.so` in-tree with nvcc for sm_100a.

    python -m paper_2003_07989_b200.build [--force] [--verbose]

The sources are csrc/*.cu (hand-written CUDA); the only public header is
include/rips.h.  The .so is git-ignored but travels to the GPU box with the tree.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "librips_b200.so")
SOURCES = ["rips.cu", "radix_sort.cu", "stage1.cu", "stage2.cu", "dim0.cu", "init.cu", "reduce.cu", "sparse.cu"]
HEADERS = ["common.cuh", "kernels.cuh", "apparent.cuh", "radix_sort.cuh", os.path.join("..", "..", "include", "rips.h")]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA path cannot be built (there is no CPU fallback)")
    return exe


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


STRESS_LIB = os.path.join(HERE, "librips_b200_stress.so")
STRESS_FLAGS = ["-DRIPS_STRESS", "-DRIPS_SORT_THREADS=256", "-DRIPS_SORT_IPT=2", "-DRIPS_SORT_MIN_BLOCKS=3", "-DRIPS_SORT_RANK_BATCH=2"]


def _compile(out: str, extra, verbose: bool) -> None:
    tmp = out + f".{os.getpid()}.tmp"
    cmd = [nvcc(), "--threads", "0", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC,-O3", "-Xcompiler", "-Wall"] + list(extra) + \
          ["-o", tmp] + [os.path.join(CSRC, f) for f in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas")
        cmd.insert(2, "-v")
    subprocess.check_call(cmd)
    os.replace(tmp, out)


def build_all(force: bool = False) -> None:
    """The product library and the stress variant, compiled side by side."""
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=2) as ex:
        a, b = ex.submit(build, force), ex.submit(build_stress, force)
        a.result(); b.result()


def _stale(out: str) -> bool:
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        _compile(LIB, [], verbose)
    return LIB


def build_stress(force: bool = False) -> str:
    """The same sources with -DRIPS_STRESS: sort tiles of 512 records, short chunks in compact mode, pseudo-random
    delays in front of every publication of the chained scans and of the lock-free reduction.  Test infrastructure
    (tests/test_gpu_parity.py::test_stress_build): same C ABI, same results, different schedules."""
    if force or _stale(STRESS_LIB):
        _compile(STRESS_LIB, STRESS_FLAGS, False)
    return STRESS_LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
    if "--stress" in sys.argv:
        print(build_stress(force="--force" in sys.argv))
