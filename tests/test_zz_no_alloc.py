"""heal_gemm_static: the entry point that allocates nothing (scratch = the hi/lo planes of A in a static device array inside
the library, include/heal.h).  Collected last on purpose (pytest -x): a failure here hides no other test.
Passes alone in a fresh process (then heal_gemm_static is the FIRST call into the library and also sets it up without
cudaMalloc) and after the other GPU tests (library already initialised)."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hb():
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    from paper_2606_21023_b200 import binding
    binding.lib()
    return binding


def _inputs(M, N, K, seed):
    gen = torch.Generator(device="cuda")
    gen.manual_seed(seed)
    A = torch.randn(M, K, device="cuda", generator=gen)
    A[:, 3] *= 40.0                                    # an outlier channel, as in the activations of the paper's models
    W = (torch.randn(K, N, device="cuda", generator=gen) * 0.02).half()
    return A, W


def test_static_scratch_matches_heal_gemm_two_calls_in_a_row(hb):
    """Two calls in a row (the second one smaller, so the array still holds the first call's planes beyond what it rewrites),
    each against the existing path: bit-identical, which is inside every tolerance the parity tests use (element-wise bound
    vs the oracle's O3, normwise 2e-6 vs FP64)."""
    shapes = [(48, 1032, 4096 + 72, hb.MODE_2P), (5, 520, 1100 - 4, hb.MODE_2P), (64, 2056, 2048, hb.MODE_1P)]
    data = [_inputs(M, N, K, 100 + i) for i, (M, N, K, _) in enumerate(shapes)]
    torch.cuda.synchronize()
    got = []
    for (A, W), (M, N, K, mode) in zip(data, shapes):
        C = torch.full((M, N), float("nan"), device="cuda")
        got.append((C, A, W, mode))
    # the new entry point first: in a fresh process this is the first call into the library
    for C, A, W, mode in got:
        hb.heal_gemm_static(A, W, mode, C=C)
    torch.cuda.synchronize()
    assert "smallm" in hb.last_kernel()
    for C, A, W, mode in got:
        ref = hb.heal_gemm(A, W, mode)
        torch.cuda.synchronize()
        assert torch.isfinite(C).all()
        assert torch.equal(C, ref)
        np.testing.assert_allclose(C.cpu().numpy(), ref.cpu().numpy(), rtol=0, atol=0)
    # the same call twice in a row gives the same bits (nothing stale is read), also through the N x K weight layout
    C0, A, W, mode = got[0]
    again = hb.heal_gemm_static(A, W, mode)
    nk = hb.heal_gemm_static(A, W.t().contiguous(), mode | hb.B_NK | hb.B_STATIC)
    torch.cuda.synchronize()
    assert torch.equal(again, C0) and torch.equal(nk, C0)
    # no allocation: the device's free memory does not move over further calls (the module and its kernels are loaded by now) ...
    Cl, Al, Wl, model = got[1]
    out = torch.empty_like(Cl)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for C, A, W, mode in got:
        hb.heal_gemm_static(A, W, mode, C=C)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    # ... and the call is legal under a global-mode stream capture, where cudaMalloc is not
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s, capture_error_mode="global"):
            hb.heal_gemm_static(Al, Wl, model, C=out)
        out.zero_()
        g.replay()
        g.replay()
    s.synchronize()
    assert torch.equal(out, Cl)


def test_static_scratch_limits_and_errors(hb):
    A = torch.zeros((65, 64), device="cuda")
    W = torch.zeros((64, 16), dtype=torch.float16, device="cuda")
    W32 = torch.zeros((64, 16), device="cuda")
    C = torch.zeros((65, 16), device="cuda")
    raw = hb.heal_gemm_static_raw
    ERR_MODE, ERR_WS = 4, 6
    assert raw(65, 16, 64, A.data_ptr(), 64, W.data_ptr(), 16, C.data_ptr(), 16, hb.MODE_2P) == ERR_WS           # M > 64
    assert raw(8, 16, 64, A.data_ptr(), 64, W32.data_ptr(), 16, C.data_ptr(), 16, 3) == ERR_MODE                  # FP32 weights
    assert raw(8, 16, 64, A.data_ptr(), 64, W.data_ptr(), 16, C.data_ptr(), 16, hb.MODE_2P | hb.LO_SCALED) == ERR_MODE
    assert raw(8, 16, 64, A.data_ptr(), 64, W.data_ptr(), 16, C.data_ptr(), 16, hb.MODE_2P | hb.EPI_ACCUMULATE) == ERR_MODE
    # planes beyond the static array: 64 x 40000 x 2 B x 2 planes > 8 MiB (rejected before any pointer is touched)
    K = 40000
    assert 2 * 64 * K * 2 > hb.STATIC_SCRATCH_BYTES
    assert raw(64, 16, K, A.data_ptr(), K, W.data_ptr(), 16, C.data_ptr(), 16, hb.MODE_2P) == ERR_WS
    assert raw(0, 16, 64, None, 64, None, 16, None, 16, hb.MODE_2P) == 0                                          # empty problem
    # K == 0: zero fill
    C.fill_(7.0)
    assert raw(8, 16, 0, None, 0, None, 16, C.data_ptr(), 16, hb.MODE_2P) == 0
    torch.cuda.synchronize()
    assert torch.all(C[:8] == 0) and torch.all(C[8:] == 7.0)
