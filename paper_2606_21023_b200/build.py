"""Build libheal.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_21023_b200.build [--force] [-v] [--trace]

--trace builds libheal_trace.so instead: the same sources with -DHEAL_TRACE (%globaltimer phase stamps in the small-M kernel, wait
counters in the CTA-pair kernel), used only by `bench.py --trace`; the product library has none of it.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libheal.so")
TRACE_LIB_PATH = os.path.join(_HERE, "libheal_trace.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "--split-compile", "0"]     # parallel back end: 2m20 -> 1m


def _sources():
    return sorted(glob.glob(os.path.join(_CSRC, "*.cu")))


def _deps():
    return _sources() + glob.glob(os.path.join(_CSRC, "*.cuh")) + glob.glob(os.path.join(_CSRC, "*.h")) + \
        [os.path.join(_HERE, "..", "include", "heal.h")]


def build(force: bool = False, verbose: bool = False, trace: bool = False) -> str:
    out = TRACE_LIB_PATH if trace else LIB_PATH
    if not force and os.path.exists(out) and \
            os.path.getmtime(out) >= max(os.path.getmtime(p) for p in _deps()):
        return out
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = out + ".tmp%d" % os.getpid()
    cmd = [nvcc] + NVCC_FLAGS + (["-DHEAL_TRACE"] if trace else []) + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + _sources()
    subprocess.check_call(cmd)
    os.replace(tmp, out)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv, trace="--trace" in sys.argv))
