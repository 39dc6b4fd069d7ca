"""Seeded synthetic inputs for the HEAL compensated-GEMM path (harness code).

Shared by the oracle-side tests and the CUDA-side tests/bench; contains none of the method's
arithmetic (see gen.c).  Shapes and value structure follow BASELINE.json's configs and
PAPER.md:201 (activations O(1), max abs < 1024, outliers in 0.1 %-1 % of *fixed channels*);
the recipe is written out in DESIGN.md "Input recipe".
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libhealinputs.so")
_lib = None

TENSOR_A = 1
TENSOR_B = 2


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _L():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        i64, u64, vp, d = ctypes.c_int64, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_double
        L.heal_inputs_fill.restype = None
        L.heal_inputs_fill.argtypes = [vp, i64, i64, i64, i64, u64, u64, ctypes.c_int, d, d, vp, i64, d,
                                       ctypes.c_int]
        L.heal_inputs_outlier_cols.restype = None
        L.heal_inputs_outlier_cols.argtypes = [vp, i64, i64, u64, u64]
        _lib = L
    return _lib


def outlier_cols(ncols: int, seed: int = 0, tensor_id: int = TENSOR_A, n: int | None = None) -> np.ndarray:
    """ceil(ncols/1000) fixed outlier channels (0.1 % of channels)."""
    n = math.ceil(ncols / 1000) if n is None else n
    cols = np.empty(n, np.int64)
    _L().heal_inputs_outlier_cols(cols.ctypes.data, n, ncols, seed, tensor_id)
    return cols


def fill(out: np.ndarray, row0: int = 0, seed: int = 0, tensor_id: int = TENSOR_A, dist: str = "normal",
         p0: float = 1.0, p1: float = 0.0, scale_cols=None, factor: float = 1.0) -> np.ndarray:
    """Fill a 2-D float32 / float16 array (unit inner stride) in place; rows row0.. of the tensor."""
    assert out.ndim == 2 and out.strides[1] == out.itemsize
    as16 = {np.dtype(np.float32): 0, np.dtype(np.float16): 1, np.dtype(np.uint16): 1}[out.dtype]
    sc = None if scale_cols is None else np.ascontiguousarray(np.asarray(scale_cols, np.int64))
    _L().heal_inputs_fill(out.ctypes.data, out.strides[0] // out.itemsize, row0, out.shape[0], out.shape[1],
                          seed, tensor_id, {"normal": 0, "uniform": 1}[dist], p0, p1,
                          None if sc is None else sc.ctypes.data, 0 if sc is None else sc.size, factor, as16)
    return out


def activations(M: int, K: int, seed: int = 0, dist: str = "normal", outliers: bool = False,
                row0: int = 0, ld: int | None = None, tensor_id: int = TENSOR_A) -> np.ndarray:
    """FP32 activations (M, K): N(0,1) or U(-1,1); optional x50 outlier channels."""
    ld = K if ld is None else ld
    buf = np.zeros((M, ld), np.float32)
    out = buf[:, :K]
    p0, p1 = (1.0, 0.0) if dist == "normal" else (-1.0, 1.0)
    sc = outlier_cols(K, seed, tensor_id) if outliers else None
    return fill(out, row0, seed, tensor_id, dist, p0, p1, sc, 50.0)


def weights_f16(K: int, N: int, seed: int = 0, sigma: float = 0.02, nk: bool = False,
                ld: int | None = None, tensor_id: int = TENSOR_B) -> np.ndarray:
    """FP16 weights N(0, sigma^2): (K, N) row-major, or the same matrix stored (N, K) if nk."""
    if nk:
        w = weights_f16(K, N, seed, sigma, False, None, tensor_id)
        ld = K if ld is None else ld
        buf = np.zeros((N, ld), np.float16)
        buf[:, :K] = w.T
        return buf[:, :K]
    ld = N if ld is None else ld
    buf = np.zeros((K, ld), np.float16)
    return fill(buf[:, :N], 0, seed, tensor_id, "normal", sigma)


def weights_f32(K: int, N: int, seed: int = 0, dist: str = "uniform", sigma: float = 1.0, nk: bool = False,
                ld: int | None = None, tensor_id: int = TENSOR_B) -> np.ndarray:
    """FP32 second operand (three-product mode): U(-1,1) or N(0, sigma^2); (K, N) or (N, K)."""
    p0, p1 = (sigma, 0.0) if dist == "normal" else (-1.0, 1.0)
    if nk:
        w = weights_f32(K, N, seed, dist, sigma, False, None, tensor_id)
        ld = K if ld is None else ld
        buf = np.zeros((N, ld), np.float32)
        buf[:, :K] = w.T
        return buf[:, :K]
    ld = N if ld is None else ld
    buf = np.zeros((K, ld), np.float32)
    return fill(buf[:, :N], 0, seed, tensor_id, dist, p0, p1)


def integers(rows: int, cols: int, lo: int, hi: int, seed: int = 0, tensor_id: int = 7,
             dtype=np.float32) -> np.ndarray:
    """Integer-valued matrix with entries uniform in [lo, hi] (exact-regime tests)."""
    u = np.zeros((rows, cols), np.float32)
    fill(u, 0, seed, tensor_id, "uniform", 0.0, 1.0)
    v = np.floor(u.astype(np.float64) * (hi - lo + 1)).astype(np.int64) + lo
    return np.clip(v, lo, hi).astype(dtype)
