"""Thin ctypes binding over libheal.so (include/heal.h).  Argument marshalling only: every step
of the path (split, tcgen05 MMAs, epilogue) runs in the CUDA kernels behind the C ABI.  torch is
used for device memory and streams.  There is no fallback: if libheal.so is missing or the device
is not sm_100 the calls raise.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libheal.so")

MODE_1P, MODE_2P, MODE_3P, MODE_4P = 1, 2, 3, 4
B_NK = 0x10
B_STATIC = 0x20
LO_SCALED = 0x40
EPI_SILU_MUL = 0x80
EPI_ACCUMULATE = 0x100
FUSE_SPLIT = 0x200
LO_SHIFT = 10
K_SEGMENT = 512

_lib = None


class HealError(RuntimeError):
    pass


def lib():
    """Load libheal.so (built by build.py / __graft_entry__.build()); fail loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise HealError(f"{LIB_PATH} not found: run `python -m paper_2606_21023_b200.build` "
                            "(there is no CPU or library fallback)")
        L = ctypes.CDLL(LIB_PATH)
        i64, vp, u32, ci = ctypes.c_int64, ctypes.c_void_p, ctypes.c_uint32, ctypes.c_int
        L.heal_gemm.restype = ci
        L.heal_gemm.argtypes = [i64, i64, i64, vp, i64, vp, i64, vp, i64, u32, vp]
        L.heal_gemm_static.restype = ci
        L.heal_gemm_static.argtypes = [i64, i64, i64, vp, i64, vp, i64, vp, i64, u32, vp]
        L.heal_gemm_host.restype = ci
        L.heal_gemm_host.argtypes = [i64, i64, i64, vp, i64, vp, i64, vp, i64, u32, vp]
        L.heal_gemm_host_act.restype = ci
        L.heal_gemm_host_act.argtypes = [i64, i64, i64, vp, i64, vp, i64, vp, i64, u32, vp]
        L.heal_split.restype = ci
        L.heal_split.argtypes = [i64, i64, vp, i64, vp, vp, i64, vp]
        L.heal_split_scaled.restype = ci
        L.heal_split_scaled.argtypes = [i64, i64, vp, i64, vp, vp, i64, ctypes.c_int32, vp]
        L.heal_rmsnorm_split.restype = ci
        L.heal_rmsnorm_split.argtypes = [i64, i64, vp, i64, vp, ctypes.c_float, vp, vp, i64, vp, i64, vp]
        L.heal_gemm_presplit.restype = ci
        L.heal_gemm_presplit.argtypes = [i64, i64, i64, vp, vp, i64, vp, vp, i64, vp, i64, u32, vp]
        i32 = ctypes.c_int32
        L.heal_gemm_ex.restype = ci
        L.heal_gemm_ex.argtypes = [i64, i64, i64, vp, i64, vp, i64, vp, i64, vp, vp, i64, i32, u32, vp]
        L.heal_gemm_presplit_ex.restype = ci
        L.heal_gemm_presplit_ex.argtypes = [i64, i64, i64, vp, vp, i64, vp, vp, i64, vp, i64, vp, vp, i64, i32, u32, vp]
        L.heal_workspace_size.restype = ctypes.c_size_t
        L.heal_workspace_size.argtypes = [i64, i64, i64, u32]
        L.heal_set_workspace.restype = ci
        L.heal_set_workspace.argtypes = [vp, ctypes.c_size_t]
        L.heal_debug_force_kernel.restype = ci
        L.heal_debug_force_kernel.argtypes = [ci]
        L.heal_launch_count.restype = ctypes.c_uint64
        L.heal_version.restype = ci
        L.heal_last_cuda_error.restype = ci
        L.heal_last_kernel.restype = ctypes.c_char_p
        L.heal_status_string.restype = ctypes.c_char_p
        L.heal_status_string.argtypes = [ci]
        _lib = L
    return _lib


def _check(st: int):
    if st != 0:
        L = lib()
        raise HealError(f"{L.heal_status_string(st).decode()} (status {st}, cudaError {L.heal_last_cuda_error()})")


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _ld(t: torch.Tensor) -> int:
    assert t.dim() == 2 and (t.shape[1] <= 1 or t.stride(1) == 1), "row-major with unit inner stride"
    return t.stride(0) if t.shape[0] > 1 else max(t.stride(0), t.shape[1])


def status_string(st: int) -> str:
    return lib().heal_status_string(st).decode()


def version() -> int:
    return lib().heal_version()


def debug_force_kernel(which: int):
    """0 auto, 1 large-M kernels only, 2 small-M for M <= 64, 3 single-CTA large-M kernel (debug)."""
    _check(lib().heal_debug_force_kernel(which))


def last_kernel() -> str:
    return lib().heal_last_kernel().decode()


def launch_count() -> int:
    return int(lib().heal_launch_count())


def workspace_size(M: int, N: int, K: int, mode: int) -> int:
    return int(lib().heal_workspace_size(M, N, K, mode))


def set_workspace(buf: torch.Tensor | None):
    if buf is None:
        _check(lib().heal_set_workspace(None, 0))
    else:
        _check(lib().heal_set_workspace(ctypes.c_void_p(buf.data_ptr()), buf.numel() * buf.element_size()))


def heal_gemm(A: torch.Tensor, B: torch.Tensor, mode: int = MODE_2P, C: torch.Tensor | None = None, stream=None):
    """C = A.B through heal_gemm (device tensors).  A fp32 (M,K); B fp16 (1P/2P) or fp32 (3P/4P),
    (K,N), or (N,K) with mode | B_NK.  Returns C fp32 (M,N)."""
    assert A.is_cuda and B.is_cuda and A.dtype == torch.float32
    nprod = mode & 0xF
    assert B.dtype == (torch.float32 if nprod >= 3 else torch.float16)
    M, K = A.shape
    N = B.shape[0] if mode & B_NK else B.shape[1]
    assert (B.shape[1] if mode & B_NK else B.shape[0]) == K
    if C is None:
        C = torch.empty((M, _n_out(N, mode)), dtype=torch.float32, device=A.device)
    _check(lib().heal_gemm(M, N, K, A.data_ptr(), _ld(A), B.data_ptr(), _ld(B), C.data_ptr(), _ld(C), mode,
                           _stream(stream)))
    return C


STATIC_SCRATCH_BYTES = 8 << 20
STATIC_MAX_M = 64


def heal_gemm_static_raw(M, N, K, A_ptr, lda, B_ptr, ldb, C_ptr, ldc, mode, stream=None) -> int:
    """Status code of heal_gemm_static, no exception (for error-path tests)."""
    return lib().heal_gemm_static(M, N, K, A_ptr, lda, B_ptr, ldb, C_ptr, ldc, mode, _stream(stream))


def heal_gemm_static(A: torch.Tensor, B: torch.Tensor, mode: int = MODE_2P, C: torch.Tensor | None = None, stream=None):
    """C = A.B through heal_gemm_static: the entry point that allocates nothing (scratch in a static device array of
    STATIC_SCRATCH_BYTES inside the library; M <= STATIC_MAX_M, FP16 weights, 1P/2P).  Calls that overlap on the GPU race."""
    assert A.is_cuda and B.is_cuda and A.dtype == torch.float32 and B.dtype == torch.float16
    M, K = A.shape
    N = B.shape[0] if mode & B_NK else B.shape[1]
    assert (B.shape[1] if mode & B_NK else B.shape[0]) == K
    if C is None:
        C = torch.empty((M, N), dtype=torch.float32, device=A.device)
    _check(lib().heal_gemm_static(M, N, K, A.data_ptr(), _ld(A), B.data_ptr(), _ld(B), C.data_ptr(), _ld(C), mode,
                                  _stream(stream)))
    return C


def _n_out(N: int, mode: int) -> int:
    """Output columns: N, or N/2 with the SiLU-mul epilogue ((gate, up) column pairs -> one activation)."""
    return N // 2 if mode & EPI_SILU_MUL else N


def _planes(M, N, device):
    ld = (N + 7) // 8 * 8
    return (torch.empty((M, ld), dtype=torch.float16, device=device)[:, :N],
            torch.empty((M, ld), dtype=torch.float16, device=device)[:, :N])


def heal_gemm_ex(A: torch.Tensor, B: torch.Tensor, mode: int = MODE_2P, C: torch.Tensor | None = None, want_c: bool = True,
                 want_planes: bool = True, scale_exp: int = 0, C_hi=None, C_lo=None, stream=None):
    """heal_gemm with the extended epilogue: returns (C or None, C_hi or None, C_lo or None); every output is the
    result times 2^-scale_exp, the planes are its hi/lo split for a following heal_gemm_presplit."""
    assert A.is_cuda and B.is_cuda and A.dtype == torch.float32
    M, K = A.shape
    N = B.shape[0] if mode & B_NK else B.shape[1]
    if C is None and want_c:
        C = torch.empty((M, _n_out(N, mode)), dtype=torch.float32, device=A.device)
    if want_planes and C_hi is None:
        C_hi, C_lo = _planes(M, _n_out(N, mode), A.device)
    p = lambda t: None if t is None else t.data_ptr()
    _check(lib().heal_gemm_ex(M, N, K, A.data_ptr(), _ld(A), B.data_ptr(), _ld(B), p(C), 0 if C is None else _ld(C),
                              p(C_hi), p(C_lo), 0 if C_hi is None else _ld(C_hi), scale_exp, mode, _stream(stream)))
    return C, C_hi, C_lo


def heal_gemm_presplit_ex(A_hi, A_lo, B_hi, B_lo, mode: int, C: torch.Tensor | None = None, want_c: bool = True,
                          want_planes: bool = True, scale_exp: int = 0, C_hi=None, C_lo=None, stream=None):
    """heal_gemm_presplit with the extended epilogue (see heal_gemm_ex)."""
    M, K = A_hi.shape
    N = B_hi.shape[0] if mode & B_NK else B_hi.shape[1]
    if C is None and want_c:
        C = torch.empty((M, _n_out(N, mode)), dtype=torch.float32, device=A_hi.device)
    if want_planes and C_hi is None:
        C_hi, C_lo = _planes(M, _n_out(N, mode), A_hi.device)
    p = lambda t: None if t is None else t.data_ptr()
    _check(lib().heal_gemm_presplit_ex(M, N, K, p(A_hi), p(A_lo), _ld(A_hi), p(B_hi), p(B_lo), _ld(B_hi), p(C),
                                       0 if C is None else _ld(C), p(C_hi), p(C_lo), 0 if C_hi is None else _ld(C_hi),
                                       scale_exp, mode, _stream(stream)))
    return C, C_hi, C_lo


def heal_gemm_raw(M, N, K, A_ptr, lda, B_ptr, ldb, C_ptr, ldc, mode, stream_ptr=None) -> int:
    """Unchecked pass-through returning the heal_status (used by the boundary tests)."""
    return lib().heal_gemm(M, N, K, A_ptr, lda, B_ptr, ldb, C_ptr, ldc, mode, stream_ptr)


def heal_split(X: torch.Tensor, hi: torch.Tensor | None = None, lo: torch.Tensor | None = None, stream=None, lo_shift: int = 0):
    """(hi, lo) fp16 planes of the fp32 matrix X (step S); lo = r16((x - hi) * 2^lo_shift)."""
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2
    rows, cols = X.shape
    if hi is None:
        ld = (cols + 7) // 8 * 8
        hi = torch.empty((rows, ld), dtype=torch.float16, device=X.device)[:, :cols]
        lo = torch.empty((rows, ld), dtype=torch.float16, device=X.device)[:, :cols]
    assert _ld(hi) == _ld(lo)
    _check(lib().heal_split_scaled(rows, cols, X.data_ptr(), _ld(X), hi.data_ptr(), lo.data_ptr(), _ld(hi), lo_shift,
                                   _stream(stream)))
    return hi, lo


def heal_rmsnorm_split(X: torch.Tensor, gamma: torch.Tensor | None = None, eps: float = 1e-6, want_y: bool = False, stream=None):
    """RMSNorm of every row of the fp32 matrix X, split into (hi, lo) fp16 planes in the same pass (PAPER.md:76 Norm -> GEMM);
    returns (hi, lo, Y or None) where Y is the fp32 normalised matrix (only written when asked for)."""
    assert X.is_cuda and X.dtype == torch.float32 and X.dim() == 2
    rows, cols = X.shape
    hi, lo = _planes(rows, cols, X.device)
    Y = torch.empty((rows, (cols + 3) // 4 * 4), dtype=torch.float32, device=X.device)[:, :cols] if want_y else None
    _check(lib().heal_rmsnorm_split(rows, cols, X.data_ptr(), _ld(X), None if gamma is None else gamma.data_ptr(), float(eps),
                                    hi.data_ptr(), lo.data_ptr(), _ld(hi), None if Y is None else Y.data_ptr(),
                                    0 if Y is None else _ld(Y), _stream(stream)))
    return hi, lo, Y


def heal_gemm_presplit(A_hi, A_lo, B_hi, B_lo, mode: int, C: torch.Tensor | None = None, stream=None):
    """C from pre-split fp16 planes (steps G + E)."""
    M, K = A_hi.shape
    N = B_hi.shape[0] if mode & B_NK else B_hi.shape[1]
    if C is None:
        C = torch.empty((M, _n_out(N, mode)), dtype=torch.float32, device=A_hi.device)
    p = lambda t: None if t is None else t.data_ptr()
    _check(lib().heal_gemm_presplit(M, N, K, p(A_hi), p(A_lo), _ld(A_hi), p(B_hi), p(B_lo), _ld(B_hi),
                                    C.data_ptr(), _ld(C), mode, _stream(stream)))
    return C


def heal_gemm_host(A: torch.Tensor, B: torch.Tensor, mode: int = MODE_2P, C: torch.Tensor | None = None, stream=None):
    """Host-buffer variant (pinned CPU tensors in, CPU tensor out); synchronises before returning."""
    assert not A.is_cuda and not B.is_cuda and A.dtype == torch.float32
    M, K = A.shape
    N = B.shape[0] if mode & B_NK else B.shape[1]
    if C is None:
        C = torch.empty((M, N), dtype=torch.float32).pin_memory()
    _check(lib().heal_gemm_host(M, N, K, A.data_ptr(), _ld(A), B.data_ptr(), _ld(B), C.data_ptr(), _ld(C), mode,
                                _stream(stream)))
    return C


def heal_gemm_host_act(A: torch.Tensor, B: torch.Tensor, mode: int = MODE_2P, C: torch.Tensor | None = None, stream=None):
    """Inference form of the host variant: pinned CPU activations in, CPU result out, weights resident on the device."""
    assert not A.is_cuda and B.is_cuda and A.dtype == torch.float32
    M, K = A.shape
    N = B.shape[0] if mode & B_NK else B.shape[1]
    if C is None:
        C = torch.empty((M, N), dtype=torch.float32).pin_memory()
    _check(lib().heal_gemm_host_act(M, N, K, A.data_ptr(), _ld(A), B.data_ptr(), _ld(B), C.data_ptr(), _ld(C), mode,
                                    _stream(stream)))
    return C
