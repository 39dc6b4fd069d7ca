"""Pins for oracle/ (CPU only).  Each test fixes a piece of the oracle to something other than
itself: hand-computed values, exact integer arithmetic, closed forms, numpy's float64 matmul and
float16 conversions (independent library code), x86 F16C hardware conversion, and the constants
the paper prints (tests/golden/paper_constants.txt).  A dropped term, wrong sign/index or a
transposed operand in O1/O2/O3 fails at least one of them.
"""
import ctypes
import os
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden_constants():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_constants.txt")):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = float(v)
    return out


# ----------------------------------------------------------------------------- O1: plain GEMM

def test_o1_tiny_hand_values(oracle):
    # 1x1x1
    assert oracle.gemm_f64(np.array([[3.0]], np.float32), np.array([[-2.5]], np.float32))[0, 0] == -7.5
    # 2x3 . 3x4, worked by hand:
    A = np.array([[1, 2, 3], [-1, 0.5, 4]], np.float32)
    B = np.array([[1, 0, 2, -1], [0, 1, 1, 3], [2, -2, 0.5, 0]], np.float32)
    want = np.array([[7, -4, 5.5, 5], [7, -7.5, 0.5, 2.5]], np.float64)
    assert np.array_equal(oracle.gemm_f64(A, B), want)
    # same B handed over as FP16 bit patterns (all entries exactly representable)
    assert np.array_equal(oracle.gemm_f64(A, B.astype(np.float16)), want)
    # and in the paper's W^T storage (N x K)
    assert np.array_equal(oracle.gemm_f64(A, np.ascontiguousarray(B.T), b_nk=True), want)
    assert np.array_equal(oracle.gemm_f64(A, np.ascontiguousarray(B.T.astype(np.float16)), b_nk=True), want)


def test_o1_asymmetric_not_transposed(oracle):
    # 5x7x3 with a non-square, non-symmetric pattern: a transposed operand or swapped index changes it
    M, N, K = 5, 7, 3
    A = np.array([[i * 10 + k for k in range(K)] for i in range(M)], np.float32)
    B = np.array([[(k + 1) * (j - 3) for j in range(N)] for k in range(K)], np.float32)
    want = np.zeros((M, N), np.int64)
    for i in range(M):
        for j in range(N):
            for k in range(K):
                want[i, j] += int(A[i, k]) * int(B[k, j])
    assert np.array_equal(oracle.gemm_f64(A, B), want.astype(np.float64))


@pytest.mark.parametrize("M,N,K", [(17, 33, 64), (8, 40, 4096), (3, 5, 65536)])
def test_o1_integer_exact(oracle, inputs, M, N, K):
    # entries in [-8, 8]: |sum| <= 64 K < 2^53, so the double GEMM must equal the int64 GEMM exactly
    A = inputs.integers(M, K, -8, 8, seed=1)
    B = inputs.integers(K, N, -8, 8, seed=2)
    want = A.astype(np.int64) @ B.astype(np.int64)
    assert np.array_equal(oracle.gemm_f64(A, B), want.astype(np.float64))
    assert np.array_equal(oracle.gemm_f64(A, B.astype(np.float16)), want.astype(np.float64))
    Bt = np.ascontiguousarray(B.T)
    assert np.array_equal(oracle.gemm_f64(A, Bt, b_nk=True), want.astype(np.float64))


def test_o1_closed_forms(oracle):
    M, N, K = 9, 11, 300
    ones = oracle.gemm_f64(np.ones((M, K), np.float32), np.ones((K, N), np.float32))
    assert np.all(ones == K)
    A = np.repeat(np.arange(1, M + 1, dtype=np.float32)[:, None], K, 1)
    B = np.repeat(np.arange(1, N + 1, dtype=np.float32)[None, :], K, 0)
    want = K * np.outer(np.arange(1, M + 1), np.arange(1, N + 1))
    assert np.array_equal(oracle.gemm_f64(A, B), want.astype(np.float64))
    # B = I  =>  C = A exactly
    rng = np.random.default_rng(0)
    A = rng.standard_normal((M, K)).astype(np.float32)
    assert np.array_equal(oracle.gemm_f64(A, np.eye(K, dtype=np.float32)), A.astype(np.float64))
    # rank one: K = 1
    u = rng.standard_normal((M, 1)).astype(np.float32)
    v = rng.standard_normal((1, N)).astype(np.float32)
    assert np.array_equal(oracle.gemm_f64(u, v), u.astype(np.float64) * v.astype(np.float64))


def test_o1_vs_numpy_float64_matmul(oracle, inputs):
    A = inputs.activations(33, 1000, seed=3, outliers=True)
    W = inputs.weights_f16(1000, 77, seed=3)
    ref = A.astype(np.float64) @ W.astype(np.float64)           # numpy's own f16->f64 and BLAS
    got = oracle.gemm_f64(A, W)
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(A.astype(np.float64)).max() * 1000
    B = inputs.weights_f32(1000, 77, seed=4)
    ref = A.astype(np.float64) @ B.astype(np.float64)
    assert np.abs(oracle.gemm_f64(A, B) - ref).max() <= 1e-10


def test_o1_row_subset_and_strides(oracle, inputs):
    A = inputs.activations(40, 128, seed=5, ld=136)           # padded leading dimension
    W = inputs.weights_f16(128, 48, seed=5, ld=56)
    full = oracle.gemm_f64(A, W)
    rows = [0, 7, 39, 8]
    sub = oracle.gemm_f64(A, W, rows=rows)
    assert np.array_equal(sub, full[rows])
    dense = oracle.gemm_f64(np.ascontiguousarray(A), np.ascontiguousarray(W))
    assert np.array_equal(full, dense)


def test_o1_empty(oracle):
    C = oracle.gemm_f64(np.zeros((3, 0), np.float32), np.zeros((0, 4), np.float32))
    assert C.shape == (3, 4) and np.all(C == 0)          # K = 0: empty sum
    assert oracle.gemm_f64(np.zeros((0, 5), np.float32), np.zeros((5, 4), np.float32)).shape == (0, 4)


# ----------------------------------------------------------------------------- O2: r16 and split

SPECIALS = [
    (0.0, 0x0000), (-0.0, 0x8000), (1.0, 0x3c00), (-2.0, 0xc000),
    (1.0 + 2.0 ** -11, 0x3c00),              # tie -> even (down)
    (1.0 + 3 * 2.0 ** -11, 0x3c02),          # tie -> even (up)
    (1.0 + 2.0 ** -11 + 2.0 ** -23, 0x3c01),  # just above the tie
    (65504.0, 0x7bff), (65519.996, 0x7bff), (65520.0, 0x7c00), (1e9, 0x7c00), (-1e9, 0xfc00),
    (2.0 ** -14, 0x0400),                    # smallest normal
    (2.0 ** -24, 0x0001),                    # smallest subnormal
    (2.0 ** -25, 0x0000),                    # tie between 0 and 2^-24 -> even (0)
    (2.0 ** -25 * 1.0000001, 0x0001),
    (3 * 2.0 ** -25, 0x0002),                # tie between 1 and 2 (x2^-24) -> even (2)
    (2.0 ** -14 - 2.0 ** -25, 0x0400),       # rounds up across the subnormal/normal boundary
    (float("inf"), 0x7c00), (float("-inf"), 0xfc00),
]


def test_o2_round16_specials(oracle):
    for x, want in SPECIALS:
        got = int(oracle.round16(np.array([x], np.float32))[0])
        assert got == want, (x, hex(got), hex(want))
    assert (int(oracle.round16(np.array([np.nan], np.float32))[0]) & 0x7c00) == 0x7c00


def test_o2_f16_decode_exhaustive_vs_numpy(oracle):
    h = np.arange(65536, dtype=np.uint32).astype(np.uint16)
    ours = oracle.f16_to_f64(h)
    theirs = h.view(np.float16).astype(np.float64)
    assert np.array_equal(np.isnan(ours), np.isnan(theirs))
    ok = ~np.isnan(theirs)
    assert np.array_equal(ours[ok], theirs[ok])
    assert np.array_equal(np.signbit(ours[ok]), np.signbit(theirs[ok]))


def test_o2_round16_vs_numpy_random_patterns(oracle):
    rng = np.random.default_rng(11)
    bits = rng.integers(0, 2 ** 32, size=4_000_000, dtype=np.uint64).astype(np.uint32)
    # plus dense coverage of the FP16 range boundaries
    edge = np.concatenate([np.arange(0x33000000 - 4096, 0x33000000 + 4096, dtype=np.uint32),   # 2^-25
                           np.arange(0x38800000 - 4096, 0x38800000 + 4096, dtype=np.uint32),   # 2^-14
                           np.arange(0x477fe000 - 8192, 0x477fe000 + 16384, dtype=np.uint32)])  # 65504
    bits = np.concatenate([bits, edge, edge | np.uint32(0x80000000)])
    x = bits.view(np.float32)
    x = x[~np.isnan(x)]
    with np.errstate(over="ignore"):
        theirs = x.astype(np.float16).view(np.uint16)
    assert np.array_equal(oracle.round16(x), theirs)


def test_o2_round16_exhaustive_vs_f16c_hardware(oracle, tmp_path):
    """All 2^32 FP32 patterns: oracle_round16 (integer code) == x86 VCVTPS2PH (hardware RNE)."""
    if "f16c" not in open("/proc/cpuinfo").read():
        pytest.skip("no F16C on this host")
    exe = tmp_path / "pin_f16c"
    subprocess.check_call(["gcc", "-O2", "-fopenmp", "-mf16c", "-o", str(exe),
                           os.path.join(HERE, "pin_f16c.c"), os.path.join(HERE, "..", "oracle", "heal_oracle.c"),
                           "-lm"])
    out = subprocess.check_output([str(exe)], text=True)
    assert out.strip().startswith("mismatches 0 of 4294967296"), out


def test_o2_split_invariant(oracle):
    """|x - (hi + lo/2^s)| <= max(2^-23 |x|, 2^-(25+s)) for finite |x| <= 65504 (A1);
    in particular 2^-22 relative (BASELINE.json north_star) wherever lo does not underflow."""
    rng = np.random.default_rng(5)
    xs = [rng.standard_normal(1_000_000).astype(np.float32),
          rng.uniform(-1, 1, 1_000_000).astype(np.float32),
          (rng.standard_normal(300_000) * 0.02).astype(np.float32),
          (rng.standard_normal(300_000) * 50).astype(np.float32),
          rng.uniform(-65504, 65504, 300_000).astype(np.float32)]
    bits = rng.integers(0, 2 ** 32, size=2_000_000, dtype=np.uint64).astype(np.uint32).view(np.float32)
    xs.append(bits[np.isfinite(bits) & (np.abs(bits) <= 65504)])
    x = np.concatenate(xs)
    xd = x.astype(np.float64)
    for s in (0, 10, 11):
        hi, lo = oracle.split(x, s)
        rec = hi.view(np.float16).astype(np.float64) + lo.view(np.float16).astype(np.float64) / 2.0 ** s
        err = np.abs(xd - rec)
        bound = np.maximum(2.0 ** -23 * np.abs(xd), 2.0 ** -(25 + s))
        assert np.all(err <= bound), (s, float((err / bound).max()))
        big = np.abs(xd) >= 2.0 ** (-3 - s)
        assert np.all(err[big] <= 2.0 ** -22 * np.abs(xd[big]))
        # hi is r16(x) and lo is r16 of the exact residual (numpy's conversions as the referee)
        assert np.array_equal(hi, x.astype(np.float16).view(np.uint16))
        res = (xd - hi.view(np.float16).astype(np.float64)) * 2.0 ** s
        with np.errstate(over="ignore"):
            want_lo = res.astype(np.float32).astype(np.float16).view(np.uint16)
        assert np.array_equal(res.astype(np.float32).astype(np.float64), res)   # residual is FP32-exact
        assert np.array_equal(lo, want_lo)


def test_o2_paper_constants(oracle):
    g = _golden_constants()
    # FP16 carries 10 explicit significand bits: the gap above 1.0 is 2^-10 ...
    one_up = oracle.f16_to_f64(np.array([0x3c01], np.uint16))[0] - 1.0
    assert one_up == 2.0 ** -g["fp16_significand_bits"]
    # ... which is the TF32 epsilon the paper prints to its 3 digits,
    assert abs(one_up - g["tf32_eps"]) < 0.005e-4
    # and FP32's epsilon is 2^-23 to the printed 3 digits.
    assert abs(2.0 ** -g["fp32_significand_bits"] - g["fp32_eps"]) < 0.005e-7
    # max |activation| < 1024 uses "less than 1/64 of the representable FP16 range"
    fp16_max = oracle.f16_to_f64(np.array([0x7bff], np.uint16))[0]
    assert fp16_max == 65504.0 and g["act_abs_max"] / fp16_max < 1.0 / 64 + 1e-4
    # the dual-FP16 pair (lo scaled by 2^10) emulates >= 20 fractional bits
    x = np.random.default_rng(1).uniform(1, 2, 100000).astype(np.float32)
    hi, lo = oracle.split(x, int(g["lo_scale_log2"]))
    rec = hi.view(np.float16).astype(np.float64) + lo.view(np.float16).astype(np.float64) / 2.0 ** g["lo_scale_log2"]
    assert np.abs(rec - x.astype(np.float64)).max() <= 2.0 ** -(g["dual_fp16_fraction_bits"] + 1)


# ----------------------------------------------------------------------------- O3: Eq. 10 exactly

def test_o3_integers_small_hi_only(oracle, inputs):
    A = inputs.integers(13, 96, -8, 8, seed=1)
    B = inputs.integers(96, 21, -8, 8, seed=2)
    want = (A.astype(np.int64) @ B.astype(np.int64)).astype(np.float64)
    for n_prod, Bx in ((1, B.astype(np.float16)), (2, B.astype(np.float16)), (3, B), (4, B)):
        assert np.array_equal(oracle.gemm_split(A, Bx, n_prod), want)


def test_o3_lo_exercising_integers(oracle, inputs):
    """Entries in [2049, 8191] are not FP16 numbers (FP16 is exact only up to 2048) but hi + lo = a
    exactly, so the two-product sum equals the integer GEMM and one product alone does not."""
    M, N, K = 9, 14, 200
    mag = inputs.integers(M, K, 2049, 8191, seed=3)
    sgn = inputs.integers(M, K, 0, 1, seed=4) * 2 - 1
    A = (mag * sgn).astype(np.float32)
    hi, lo = oracle.split(A)
    assert np.any(lo.view(np.float16) != 0)
    assert np.array_equal(hi.view(np.float16).astype(np.float64) + lo.view(np.float16).astype(np.float64), A)
    B = inputs.integers(K, N, -1, 1, seed=5)
    want = (A.astype(np.int64) @ B.astype(np.int64)).astype(np.float64)
    assert np.array_equal(oracle.gemm_split(A, B.astype(np.float16), 2), want)
    assert not np.array_equal(oracle.gemm_split(A, B.astype(np.float16), 1), want)
    # three-product: lo only in A, lo only in B (roles swapped)
    assert np.array_equal(oracle.gemm_split(A, B, 3), want)
    assert np.array_equal(oracle.gemm_split(np.ascontiguousarray(B.T), np.ascontiguousarray(A.T), 3), want.T)


def test_o3_dropped_lo_lo_term(oracle, inputs):
    """lo in both operands: 3P = integer GEMM - sum lo_a lo_b (the dropped term); 4P = integer GEMM."""
    M, N, K = 6, 10, 128
    vals = np.array([2049, -2049, 4098, -4098, 0], np.float32)
    A = vals[inputs.integers(M, K, 0, 4, seed=6).astype(np.int64)]
    B = vals[inputs.integers(K, N, 0, 4, seed=7).astype(np.int64)]
    full = A.astype(np.int64) @ B.astype(np.int64)
    lo_a = np.sign(A) * np.where(np.abs(A) == 2049, 1, np.where(np.abs(A) == 4098, 2, 0))
    lo_b = np.sign(B) * np.where(np.abs(B) == 2049, 1, np.where(np.abs(B) == 4098, 2, 0))
    dropped = lo_a.astype(np.int64) @ lo_b.astype(np.int64)
    assert np.any(dropped != 0)
    assert np.array_equal(oracle.gemm_split(A, B, 4), full.astype(np.float64))
    assert np.array_equal(oracle.gemm_split(A, B, 3), (full - dropped).astype(np.float64))


def test_o3_matches_numpy_on_split_planes(oracle, inputs):
    """O3 = (hi + lo/2^s) planes pushed through numpy's float64 matmul (planes from numpy float16)."""
    A = inputs.activations(12, 300, seed=8, outliers=True)
    B = inputs.weights_f32(300, 20, seed=8)
    W = inputs.weights_f16(300, 20, seed=8)
    f = lambda u: u.view(np.float16).astype(np.float64)
    for s in (0, 10):
        ah, al = oracle.split(A, s)
        bh, bl = oracle.split(B, s)
        sc = 2.0 ** -s
        assert np.allclose(oracle.gemm_split(A, W, 2, s), (f(ah) + f(al) * sc) @ W.astype(np.float64),
                           rtol=0, atol=1e-12)
        want3 = f(ah) @ f(bh) + f(ah) @ (f(bl) * sc) + (f(al) * sc) @ f(bh)
        assert np.allclose(oracle.gemm_split(A, B, 3, s), want3, rtol=0, atol=1e-11)
        assert np.allclose(oracle.gemm_split(A, B, 1, s), f(ah) @ f(bh), rtol=0, atol=1e-11)
        Wt = np.ascontiguousarray(W.T)
        assert np.array_equal(oracle.gemm_split(A, Wt, 2, s, b_nk=True), oracle.gemm_split(A, W, 2, s))


def test_o3_close_to_o1_and_ordering(oracle, inputs):
    """Algorithmic error of Eq. 10: compensated << single FP16 cast, and bounded
    by the split invariant: |O3 - O1| <= 2^-22 sum_k |a||b| (2P), 2 * 2^-22 (+lo.lo 2^-22) (3P)."""
    A = inputs.activations(16, 4096, seed=0, outliers=True)
    W = inputs.weights_f16(4096, 24, seed=0)
    o1 = oracle.gemm_f64(A, W)
    absprod = np.abs(A.astype(np.float64)) @ np.abs(W.astype(np.float64))
    e2 = np.abs(oracle.gemm_split(A, W, 2) - o1)
    e1 = np.abs(oracle.gemm_split(A, W, 1) - o1)
    assert np.all(e2 <= 2.0 ** -22 * absprod)
    assert np.linalg.norm(e2) < 1e-3 * np.linalg.norm(e1)
    B = inputs.weights_f32(4096, 24, seed=0)
    o1 = oracle.gemm_f64(A, B)
    absprod = np.abs(A.astype(np.float64)) @ np.abs(B.astype(np.float64))
    e3 = np.abs(oracle.gemm_split(A, B, 3) - o1)
    assert np.all(e3 <= 3 * 2.0 ** -22 * absprod)
    # normwise metric of the acceptance test, on config-0-shaped inputs (SURVEY.md model: ~4.8e-9)
    A0 = inputs.activations(64, 256, seed=0)
    B0 = inputs.weights_f32(256, 256, seed=0, dist="normal")
    C3 = oracle.gemm_split(A0, B0, 3).astype(np.float32)
    e = oracle.normwise_error(C3, oracle.gemm_f64(A0, B0), A0, B0)
    assert e < 5e-8      # includes the final FP32 rounding of C3


def test_metric_definition(oracle):
    A = np.array([[3.0, 4.0]], np.float32)                      # ||A||_F = 5
    B = np.array([[1.0], [2.0]], np.float32)                    # ||B||_F = sqrt(5)
    Cref = oracle.gemm_f64(A, B)                                # 11
    C = np.array([[11.5]], np.float32)
    assert abs(oracle.normwise_error(C, Cref, A, B) - 0.5 / (5 * np.sqrt(5))) < 1e-15
    assert abs(oracle.normwise_error(C, Cref, A, B.astype(np.float16)) - 0.5 / (5 * np.sqrt(5))) < 1e-15


def test_metric_rows_list_and_padded_operands_vs_numpy(oracle):
    """The sampled-row form of the acceptance metric -- the one every full-size gate (configs[2], [3], [4], bench.py's
    normwise_err_vs_fp64) goes through: a `rows` list in non-ascending order with a repeat, C inside a buffer with
    ldc > N, FP16 B inside a buffer with ld > cols, FP32 A with lda > K.  Pinned against numpy.linalg.norm in float64
    (an independent evaluation of e = ||C_S - Cref||_F / (||A_S||_F ||B||_F), BASELINE.json north_star); a dropped
    row index, a row/column stride mix-up or padding leaking into a norm changes the value by far more than 1e-14."""
    rng = np.random.default_rng(5)
    M, N, K = 23, 24, 40
    Abuf = rng.standard_normal((M, K + 4)).astype(np.float32)
    A = Abuf[:, :K]
    Bbuf = (rng.standard_normal((K, N + 8)) * 0.02).astype(np.float16)
    Bbuf[:, N:] = np.float16(7.0)                               # padding must not enter ||B||_F
    B = Bbuf[:, :N]
    Cbuf = np.full((M, N + 5), 1e3, np.float32)                 # padding must not enter the difference
    C = Cbuf[:, :N]
    exact = A.astype(np.float64) @ B.astype(np.float64)
    C[:] = (exact + 1e-3 * rng.standard_normal((M, N))).astype(np.float32)
    rows = [17, 3, 22, 0, 9, 3, 11]
    ref = oracle.gemm_f64(A, B, rows=rows)
    assert np.allclose(ref, exact[rows], rtol=1e-13, atol=1e-13)
    want = np.linalg.norm(C[rows].astype(np.float64) - exact[rows]) / (
        np.linalg.norm(A[rows].astype(np.float64)) * np.linalg.norm(B.astype(np.float64)))
    got = oracle.normwise_error(C, ref, A, B, rows=rows)
    assert abs(got - want) <= 1e-14 * want, (got, want)
    # the same through the FP32-B form (three-product configs) and with the full-matrix call
    B32buf = rng.uniform(-1, 1, (K, N + 4)).astype(np.float32)
    B32 = B32buf[:, :N]
    ex32 = A.astype(np.float64) @ B32.astype(np.float64)
    C[:] = (ex32 * (1 + 1e-5)).astype(np.float32)
    want = np.linalg.norm(C[rows].astype(np.float64) - ex32[rows]) / (
        np.linalg.norm(A[rows].astype(np.float64)) * np.linalg.norm(B32.astype(np.float64)))
    got = oracle.normwise_error(C, oracle.gemm_f64(A, B32, rows=rows), A, B32, rows=rows)
    assert abs(got - want) <= 1e-14 * want, (got, want)
    want = np.linalg.norm(C.astype(np.float64) - ex32) / (np.linalg.norm(A.astype(np.float64)) * np.linalg.norm(B32.astype(np.float64)))
    got = oracle.normwise_error(C, oracle.gemm_f64(A, B32), A, B32)
    assert abs(got - want) <= 1e-14 * want, (got, want)
    # the raw C routines on strided data
    L = oracle.lib()
    assert abs(L.oracle_sumsq_f16(K, N, Bbuf.ctypes.data, N + 8) - float((B.astype(np.float64) ** 2).sum())) <= 1e-14 * float((B.astype(np.float64) ** 2).sum())
    assert abs(L.oracle_sumsq_f32(M, K, Abuf.ctypes.data, K + 4) - float((A.astype(np.float64) ** 2).sum())) <= 1e-13 * float((A.astype(np.float64) ** 2).sum())


# ---------------------------------------------------------------- F1-F4: steps around the GEMMs (oracle/heal_fusions.c)
def test_f1_rmsnorm_hand_values_and_invariants(oracle):
    """F1 ("Norm"; A17).  Hand-worked: x = (3, 4): mean square 12.5, so y = x / sqrt(12.5) =
    (0.6 sqrt 2, 0.8 sqrt 2); with gamma = (2, -1): (1.2 sqrt 2, -0.8 sqrt 2).  Invariants a wrong formula breaks: unit mean
    square for gamma = 1, eps = 0 (fails for LayerNorm-style mean subtraction or a sum instead of a mean), invariance under
    scaling the row (fails if eps or the 1/K is misplaced), a constant row maps to sign(c) gamma, the zero row with eps > 0 maps
    to 0, eps enters under the root (x = (1, 1), eps = 3: y = 1/2), per-row statistics and per-column gamma (fails if
    transposed), padding ignored."""
    r2 = np.sqrt(2.0)
    X = np.array([[3.0, 4.0]], np.float32)
    assert np.allclose(oracle.rmsnorm_f64(X), [[0.6 * r2, 0.8 * r2]], rtol=1e-15, atol=0)
    assert np.allclose(oracle.rmsnorm_f64(X, gamma=[2.0, -1.0]), [[1.2 * r2, -0.8 * r2]], rtol=1e-15, atol=0)
    assert np.allclose(oracle.rmsnorm_f64(np.ones((1, 2), np.float32), eps=3.0), [[0.5, 0.5]], rtol=1e-15, atol=0)
    rng = np.random.default_rng(11)
    buf = rng.standard_normal((5, 40)).astype(np.float32)
    buf[:, 37:] = 1e6                                            # padding
    Xp = buf[:, :37]
    Y = oracle.rmsnorm_f64(Xp)
    assert np.allclose((Y ** 2).mean(axis=1), 1.0, rtol=1e-14)
    assert np.allclose(oracle.rmsnorm_f64(np.ascontiguousarray(Xp) * np.float32(8.0)), Y, rtol=1e-15)      # exact power-of-two scaling
    gam = rng.standard_normal(37).astype(np.float32)
    Yg = oracle.rmsnorm_f64(Xp, gamma=gam)
    assert np.allclose(Yg, Y * gam.astype(np.float64)[None, :], rtol=1e-15)
    Xc = np.full((2, 7), -2.5, np.float32)
    assert np.allclose(oracle.rmsnorm_f64(Xc, gamma=np.arange(1, 8)), -np.arange(1, 8, dtype=np.float64)[None, :].repeat(2, 0), rtol=1e-15)
    assert np.array_equal(oracle.rmsnorm_f64(np.zeros((1, 4), np.float32), eps=1e-6), np.zeros((1, 4)))
    # rows are independent: a row with 100x the magnitude does not change its neighbour
    X2 = np.ascontiguousarray(Xp[:2]).copy()
    X2[1] *= 100
    assert np.array_equal(oracle.rmsnorm_f64(X2)[0], Y[0])


def test_f2_silu_mul_closed_forms_and_interleaving(oracle):
    """F2 ("SiLU(g) (.) u"; A18).  Closed forms: silu(0) = 0; silu(ln 3) = 3/4 ln 3 (sigmoid(ln 3) = 3/4);
    silu(-ln 3) = -1/4 ln 3; silu(x) - silu(-x) = x; large x: silu(x) -> x, silu(-x) -> 0.  Interleaving: gate is the EVEN
    column, up the ODD one (swapping them, or reading g and u from two halves of the row, fails the asymmetric cases)."""
    l3 = np.log(3.0)
    C = np.array([[0.0, 5.0, l3, 2.0, -l3, 4.0, 40.0, 0.5, -40.0, 7.0]])
    H = oracle.silu_mul_f64(C)
    assert H.shape == (1, 5)
    assert np.allclose(H[0, :3], [0.0, 0.75 * l3 * 2.0, -0.25 * l3 * 4.0], rtol=1e-15, atol=0)
    assert abs(H[0, 3] - 20.0) < 1e-14 and abs(H[0, 4]) < 1e-14
    rng = np.random.default_rng(12)
    g = rng.standard_normal((6, 9)) * 3
    Cp = np.empty((6, 18)); Cp[:, 0::2] = g; Cp[:, 1::2] = 1.0
    Cm = np.empty((6, 18)); Cm[:, 0::2] = -g; Cm[:, 1::2] = 1.0
    assert np.allclose(oracle.silu_mul_f64(Cp) - oracle.silu_mul_f64(Cm), g, rtol=1e-14, atol=1e-15)
    # u scales linearly, g does not; rows keep their place
    u = rng.standard_normal((6, 9))
    Cu = Cp.copy(); Cu[:, 1::2] = u
    assert np.allclose(oracle.silu_mul_f64(Cu), oracle.silu_mul_f64(Cp) * u, rtol=1e-15)
    assert np.array_equal(oracle.silu_mul_f64(Cu[2:3]), oracle.silu_mul_f64(Cu)[2:3])


def test_f3_gemm_dd_matches_o1_and_integers(oracle, inputs):
    """F3 = O1's definition with a double first operand: bit-identical to O1 when the doubles are FP32 values (same sums in
    the same order), exact on integer matrices, honours b_nk, row lists and padded B; asymmetric shapes catch a transposed
    operand.  F4: the residual add."""
    A = inputs.activations(9, 50, seed=3)
    W = inputs.weights_f16(50, 24, seed=3, ld=32)
    B32 = inputs.weights_f32(50, 24, seed=3, ld=28)
    Ad = A.astype(np.float64)
    assert np.array_equal(oracle.gemm_dd(Ad, W), oracle.gemm_f64(A, W))
    assert np.array_equal(oracle.gemm_dd(Ad, B32), oracle.gemm_f64(A, B32))
    rows = [7, 0, 3]
    assert np.array_equal(oracle.gemm_dd(Ad, W, rows=rows), oracle.gemm_f64(A, W)[rows])
    Wnk = inputs.weights_f16(50, 24, seed=3, nk=True)
    assert np.array_equal(oracle.gemm_dd(Ad, Wnk, b_nk=True), oracle.gemm_f64(A, W))
    Ai = inputs.integers(5, 33, -8, 8, seed=1)
    Bi = inputs.integers(33, 7, -8, 8, seed=2)
    assert np.array_equal(oracle.gemm_dd(Ai.astype(np.float64), Bi), (Ai.astype(np.int64) @ Bi.astype(np.int64)).astype(np.float64))
    # a genuinely double operand: against numpy float64 matmul
    Ah = Ad + 1e-9 * np.arange(Ad.size).reshape(Ad.shape)
    ref = Ah @ W.astype(np.float64)
    assert np.allclose(oracle.gemm_dd(Ah, W), ref, rtol=1e-13, atol=1e-14)
    Y = np.arange(18, dtype=np.float64).reshape(3, 6) * 0.25
    Xb = np.arange(24, dtype=np.float32).reshape(3, 8)
    assert np.array_equal(oracle.add_f64(Xb[:, :6], Y), Xb[:, :6].astype(np.float64) + Y)
