"""oracle/ -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes front for ``heal_oracle.c`` (plain C, FP64, gcc only): the CPU reference for HEAL's
compensated GEMM (Eq. 10; Eq. 9 PAPER.md:195 for the three-product form).
Only tests/, ``__graft_entry__.smoke()`` and bench.py's ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_2606_21023_b200``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "heal_oracle.c")
_SRC2 = os.path.join(_HERE, "heal_fusions.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile heal_oracle.c + heal_fusions.c with gcc (-O2, OpenMP, no FP contraction) into liboracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC2)):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
                               "-o", tmp, _SRC, _SRC2, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        i64, vp, ci = ctypes.c_int64, ctypes.c_void_p, ctypes.c_int
        L.oracle_f16_to_f64.restype = ctypes.c_double
        L.oracle_f16_to_f64.argtypes = [ctypes.c_uint16]
        L.oracle_round16.restype = ctypes.c_uint16
        L.oracle_round16.argtypes = [ctypes.c_float]
        L.oracle_split.restype = None
        L.oracle_split.argtypes = [i64, vp, vp, vp, ci]
        L.oracle_gemm_f64.restype = ci
        L.oracle_gemm_f64.argtypes = [i64, i64, i64, vp, i64, vp, i64, ci, ci, vp, i64, vp]
        L.oracle_gemm_split.restype = ci
        L.oracle_gemm_split.argtypes = [i64, i64, i64, vp, i64, vp, i64, ci, ci, ci, ci, vp, i64, vp]
        L.oracle_sumsq_f32.restype = ctypes.c_double
        L.oracle_sumsq_f32.argtypes = [i64, i64, vp, i64]
        L.oracle_sumsq_f16.restype = ctypes.c_double
        L.oracle_sumsq_f16.argtypes = [i64, i64, vp, i64]
        L.oracle_diff_sumsq.restype = ctypes.c_double
        L.oracle_diff_sumsq.argtypes = [i64, i64, vp, i64, vp, vp]
        L.oracle_num_threads.restype = ci
        d = ctypes.c_double
        L.oracle_rmsnorm_f64.restype = None
        L.oracle_rmsnorm_f64.argtypes = [i64, i64, vp, i64, vp, d, vp]
        L.oracle_silu_mul_f64.restype = None
        L.oracle_silu_mul_f64.argtypes = [i64, i64, vp, vp]
        L.oracle_gemm_dd.restype = ci
        L.oracle_gemm_dd.argtypes = [i64, i64, i64, vp, vp, i64, ci, ci, vp, i64, vp]
        L.oracle_add_f64.restype = None
        L.oracle_add_f64.argtypes = [i64, i64, vp, i64, vp, vp]
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def _check_a(A):
    assert A.dtype == np.float32 and A.ndim == 2
    if A.size == 0:
        return max(A.shape[1], 1)
    assert A.strides[1] == 4
    return A.strides[0] // 4


def _check_b(B):
    assert B.ndim == 2
    if B.size == 0:
        return (0 if B.dtype == np.float32 else 1), max(B.shape[1], 1)
    if B.dtype == np.float32:
        assert B.strides[1] == 4
        return 0, B.strides[0] // 4
    assert B.dtype in (np.float16, np.uint16) and B.strides[1] == 2
    return 1, B.strides[0] // 2


def _rows(rows):
    if rows is None:
        return None, 0
    r = np.ascontiguousarray(np.asarray(rows, dtype=np.int64))
    return r, r.size


def round16(x) -> np.ndarray:
    """r16(): FP32 -> binary16 bit patterns (uint16), RNE, via the oracle's integer code."""
    x = np.ascontiguousarray(np.asarray(x, dtype=np.float32))
    hi = np.empty(x.shape, np.uint16)
    lo = np.empty(x.shape, np.uint16)
    lib().oracle_split(x.size, _ptr(x), _ptr(hi), _ptr(lo), 0)
    return hi


def split(x, s: int = 0):
    """O2: (hi, lo) binary16 bit patterns (uint16) with x ~ hi + lo / 2^s."""
    x = np.ascontiguousarray(np.asarray(x, dtype=np.float32))
    hi = np.empty(x.shape, np.uint16)
    lo = np.empty(x.shape, np.uint16)
    lib().oracle_split(x.size, _ptr(x), _ptr(hi), _ptr(lo), int(s))
    return hi, lo


def f16_to_f64(h) -> np.ndarray:
    h = np.ascontiguousarray(np.asarray(h).view(np.uint16))
    out = np.empty(h.shape, np.float64)
    L = lib()
    flat_h, flat_o = h.reshape(-1), out.reshape(-1)
    for i in range(flat_h.size):
        flat_o[i] = L.oracle_f16_to_f64(int(flat_h[i]))
    return out


def gemm_f64(A, B, b_nk: bool = False, rows=None) -> np.ndarray:
    """O1: Cref = A.B in double (k ascending, one accumulator per element).

    A: float32 (M, K).  B: float32 or float16/uint16-bits, (K, N) -- or (N, K) if b_nk.
    rows: optional row indices of A; the result then has len(rows) rows.
    """
    lda = _check_a(A)
    b16, ldb = _check_b(B)
    M, K = A.shape
    N = B.shape[0] if b_nk else B.shape[1]
    assert (B.shape[1] if b_nk else B.shape[0]) == K
    r, nr = _rows(rows)
    C = np.empty(((nr if rows is not None else M), N), np.float64)
    rc = lib().oracle_gemm_f64(M, N, K, _ptr(A), lda, _ptr(B), ldb, b16, int(b_nk), _ptr(r), nr, _ptr(C))
    assert rc == 0
    return C


def gemm_split(A, B, n_prod: int, s: int = 0, b_nk: bool = False, rows=None) -> np.ndarray:
    """O3: the products the mode keeps (Eq. 10 / Eq. 9), summed exactly in double."""
    lda = _check_a(A)
    b16, ldb = _check_b(B)
    M, K = A.shape
    N = B.shape[0] if b_nk else B.shape[1]
    assert (B.shape[1] if b_nk else B.shape[0]) == K
    r, nr = _rows(rows)
    C = np.empty(((nr if rows is not None else M), N), np.float64)
    rc = lib().oracle_gemm_split(M, N, K, _ptr(A), lda, _ptr(B), ldb, b16, int(b_nk), int(n_prod), int(s),
                                 _ptr(r), nr, _ptr(C))
    assert rc == 0, rc
    return C


def fro_f32(X) -> float:
    ld = _check_a(X)
    return float(np.sqrt(lib().oracle_sumsq_f32(X.shape[0], X.shape[1], _ptr(X), ld)))


def fro_b(B) -> float:
    b16, ld = _check_b(B)
    L = lib()
    f = L.oracle_sumsq_f16 if b16 else L.oracle_sumsq_f32
    return float(np.sqrt(f(B.shape[0], B.shape[1], _ptr(B), ld)))


def normwise_error(C, Cref, A, B, rows=None) -> float:
    """e = ||C - Cref||_F / (||A||_F ||B||_F)  (BASELINE.json north_star acceptance metric).

    C: float32 (M, N) from the path under test; Cref: float64 from gemm_f64 (all rows, or the
    listed rows -- then ||A_S||_F uses the same rows of A)."""
    assert C.dtype == np.float32 and C.strides[1] == 4
    r, nr = _rows(rows)
    R = nr if rows is not None else C.shape[0]
    Cref = np.ascontiguousarray(Cref)
    d = lib().oracle_diff_sumsq(R, C.shape[1], _ptr(C), C.strides[0] // 4, _ptr(r), _ptr(Cref))
    As = A if rows is None else np.ascontiguousarray(A[np.asarray(rows)])
    return float(np.sqrt(d)) / (fro_f32(As) * fro_b(B))


def rmsnorm_f64(X, gamma=None, eps: float = 0.0) -> np.ndarray:
    """F1: RMSNorm of every row of the float32 matrix X in double ("Norm"; A17)."""
    ldx = _check_a(X)
    g = None if gamma is None else np.ascontiguousarray(np.asarray(gamma, dtype=np.float32))
    assert g is None or g.shape == (X.shape[1],)
    Y = np.empty(X.shape, np.float64)
    lib().oracle_rmsnorm_f64(X.shape[0], X.shape[1], _ptr(X), ldx, _ptr(g), float(eps), _ptr(Y))
    return Y


def silu_mul_f64(C) -> np.ndarray:
    """F2: h[j] = silu(c[2j]) * c[2j+1] on every row of the double matrix C ("SiLU(g) (.) u"; A18)."""
    C = np.ascontiguousarray(np.asarray(C, dtype=np.float64))
    assert C.ndim == 2 and C.shape[1] % 2 == 0
    H = np.empty((C.shape[0], C.shape[1] // 2), np.float64)
    lib().oracle_silu_mul_f64(C.shape[0], C.shape[1] // 2, _ptr(C), _ptr(H))
    return H


def gemm_dd(A, B, b_nk: bool = False, rows=None) -> np.ndarray:
    """F3: O1's definition for a double first operand (the next GEMM of a chain): A float64 (M, K), B as in gemm_f64."""
    A = np.ascontiguousarray(np.asarray(A, dtype=np.float64))
    b16, ldb = _check_b(B)
    M, K = A.shape
    N = B.shape[0] if b_nk else B.shape[1]
    assert (B.shape[1] if b_nk else B.shape[0]) == K
    r, nr = _rows(rows)
    C = np.empty(((nr if rows is not None else M), N), np.float64)
    rc = lib().oracle_gemm_dd(M, N, K, _ptr(A), _ptr(B), ldb, b16, int(b_nk), _ptr(r), nr, _ptr(C))
    assert rc == 0
    return C


def add_f64(X, Y) -> np.ndarray:
    """F4: the residual add X + Y, X float32, Y float64, in double."""
    ldx = _check_a(X)
    Y = np.ascontiguousarray(np.asarray(Y, dtype=np.float64))
    assert Y.shape == X.shape
    Z = np.empty(X.shape, np.float64)
    lib().oracle_add_f64(X.shape[0], X.shape[1], _ptr(X), ldx, _ptr(Y), _ptr(Z))
    return Z


def num_threads() -> int:
    return int(lib().oracle_num_threads())
