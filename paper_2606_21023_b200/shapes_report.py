"""Times every BASELINE.json config through the C ABI and prints a markdown report:
effective TFLOP/s (2MNK/t), tensor work (n_prod x that) against the dense FP16 peak, achieved HBM GB/s
for the small-M shapes, and -- as context rows on the same inputs -- cuBLAS SGEMM (TF32 off), BF16 and
FP16 GEMMs via torch.matmul.  Normwise errors vs the FP64 oracle are NOT computed here (this module
never touches oracle/); tests/test_gpu_parity.py and bench.py do that.

    python -m paper_2606_21023_b200.shapes_report > gpurun_out/shapes.md

Protocol: >= 5 warm-ups; kernels shorter than ~50 us are timed as a CUDA graph of back-to-back launches
rotating over enough distinct weight copies to exceed the 126 MB L2; longer ones as 20 back-to-back
launches; CUDA events on the launching stream; min and median of 7 repeats.  The GPU idles 1.5 s before
every measurement: these are burst figures (the 1 kW power cap pulls a hot B200 down to ~1.3-1.5 GHz; bench.py
reports the sustained regime with its clocks).
"""
from __future__ import annotations

import json
import os
import sys
import time

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from paper_2606_21023_b200 import binding as hb  # noqa: E402

L2_BYTES = 126e6
COOL_DOWN_S = 1.5


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d["bf16_tflops"], d["bf16_tflops_sustained"], d["hbm_gbs"], "measured"
    return 1590.0, 1400.0, 6650.0, "fallback"


def _time(fns, graph: bool, reps: int = 7):
    """fns: list of callables run back to back (one per weight copy); returns (min_us, med_us) per call."""
    time.sleep(COOL_DOWN_S)                  # start every measurement from an idle, un-throttled GPU
    s = torch.cuda.Stream()
    n_calls = len(fns) if graph else max(len(fns), 20 // len(fns) * len(fns))
    with torch.cuda.stream(s):
        for _ in range(2):
            for f in fns:
                f()
        s.synchronize()
        if graph:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=s):
                for f in fns:
                    f()
            run = g.replay
        else:
            def run():
                for i in range(n_calls):
                    fns[i % len(fns)]()
        run()
        s.synchronize()
        ts = []
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(s)
            run()
            e1.record(s)
            s.synchronize()
            ts.append(e0.elapsed_time(e1) * 1e3 / n_calls)
    ts.sort()
    return ts[0], ts[len(ts) // 2]


def bench_shape(name, M, N, K, nprod, dist, rows, flags=0):
    gen = torch.Generator(device="cuda")
    gen.manual_seed(1234)
    w_bytes = K * N * (4 if nprod >= 3 else 2)
    small = 2.0 * nprod * M * N * K < 5e10                 # launch-latency scale: use graphs + weight rotation
    ncopies = max(2, min(16, int(3 * L2_BYTES // w_bytes) + 1)) if small else 1
    if dist == "uniform":
        A = torch.rand(M, K, device="cuda", generator=gen) * 2 - 1
        Bs = [torch.rand(K, N, device="cuda", generator=gen) * 2 - 1 for _ in range(ncopies)]
    else:
        A = torch.randn(M, K, device="cuda", generator=gen)
        Bs = [torch.randn(K, N, device="cuda", generator=gen) * (1.0 if nprod >= 3 else 0.02) for _ in range(ncopies)]
    if nprod < 3:
        Bs = [b.half() for b in Bs]
    C = torch.empty(M, N, device="cuda")
    ws = torch.empty(max(256, hb.workspace_size(M, N, K, nprod)), dtype=torch.uint8, device="cuda")
    hb.set_workspace(ws)
    full = [(lambda b=b: hb.heal_gemm(A, b, nprod | flags, C)) for b in Bs]
    full_st = [(lambda b=b: hb.heal_gemm(A, b, nprod | flags | hb.B_STATIC, C)) for b in Bs]
    ah, al = hb.heal_split(A, lo_shift=hb.LO_SHIFT if flags & hb.LO_SCALED else 0)
    planes = [(hb.heal_split(b) if nprod >= 3 else (b, None)) for b in Bs]
    pres = [(lambda p=p: hb.heal_gemm_presplit(ah, al, p[0], p[1], nprod | flags, C)) for p in planes]
    reps = (2 if small else 1)
    t_full = _time(full * reps, small)
    t_pre = _time(pres * reps, small)
    t_st = _time(full_st * reps, small) if M <= 64 else None
    # context: cuBLAS on the same inputs
    torch.backends.cuda.matmul.allow_tf32 = False
    A16, Ab = A.half(), A.bfloat16()
    B32 = [b.float() for b in Bs]
    B16 = [b.half() for b in Bs]
    Bb = [b.bfloat16() for b in Bs]
    C16, Cb = torch.empty(M, N, device="cuda", dtype=torch.float16), torch.empty(M, N, device="cuda", dtype=torch.bfloat16)
    t_sgemm = _time([(lambda b=b: torch.matmul(A, b, out=C)) for b in B32] * reps, small, reps=3)
    t_f16 = _time([(lambda b=b: torch.matmul(A16, b, out=C16)) for b in B16] * reps, small, reps=3)
    t_bf16 = _time([(lambda b=b: torch.matmul(Ab, b, out=Cb)) for b in Bb] * reps, small, reps=3)
    hb.set_workspace(None)
    flop = 2.0 * M * N * K
    byt = K * N * 2 + M * K * 4 + M * N * 4
    burst, sust, hbm, _ = _peaks()
    st_col = "-" if t_st is None else f"{t_st[1]:.1f} ({byt / t_st[1] / 1e3:.0f} GB/s, {byt / t_st[1] / 1e3 / hbm * 100:.0f}%)"
    rows.append(f"| {name} | {M}x{N}x{K} | {nprod}P | {t_full[1]:.1f} | {st_col} | {t_pre[1]:.1f} ({t_pre[0]:.1f}) | "
                f"{flop / t_pre[1] / 1e6:.1f} | {nprod * flop / t_pre[1] / 1e6:.0f} ({nprod * flop / t_pre[1] / 1e6 / burst * 100:.0f}% / "
                f"{nprod * flop / t_pre[1] / 1e6 / 2250 * 100:.0f}%) | {byt / t_pre[1] / 1e3:.0f} ({byt / t_pre[1] / 1e3 / hbm * 100:.0f}%) | "
                f"{t_sgemm[1]:.1f} | {t_f16[1]:.1f} | {t_bf16[1]:.1f} | {'graph+rot%d' % ncopies if small else 'loop'} |")
    del Bs, B32, B16, Bb, planes
    torch.cuda.empty_cache()


def products_sweep():
    M, N, K = 2048, 14336, 4096
    gen = torch.Generator(device="cuda")
    gen.manual_seed(99)
    A = torch.randn(M, K, device="cuda", generator=gen)
    B = torch.randn(K, N, device="cuda", generator=gen) * 0.02
    ah, al = hb.heal_split(A)
    bh, bl = hb.heal_split(B)
    C = torch.empty(M, N, device="cuda")
    out = []
    steps = (N // 256) * (M // 256) * (K // 64) / 74.0            # k-tile steps per CTA pair
    for nprod, kb in ((1, 32), (2, 48), (3, 64), (4, 64)):
        t = _time([lambda: hb.heal_gemm_presplit(ah, al, bh, bl, nprod, C)], False)
        out.append(f"| {nprod}P | {t[1]:.1f} | {nprod * 2.0 * M * N * K / t[1] / 1e6:.0f} | {kb} | {kb * 1024 * steps / t[1] / 1e3:.0f} |")
    return out


def main():
    burst, sust, hbm, src = _peaks()
    rows = []
    cfgs = [("cfg0 single", 64, 256, 256, 3, "normal")]
    cfgs += [(f"cfg1 decode M={m}", m, 4096, 4096, 2, "normal") for m in (1, 8, 32)]
    cfgs += [("cfg2 MLP up/gate", 2048, 14336, 4096, 2, "normal"), ("cfg2 MLP down", 2048, 4096, 14336, 2, "normal")]
    cfgs += [(f"cfg3 square {n}", n, n, n, 3, "uniform") for n in (1024, 2048, 4096, 8192)]
    cfgs += [(f"cfg4 LM head M={m}", m, 128256, 4096, 2, "normal") for m in (1, 64, 512)]
    # beyond BASELINE.json: the other GEMM sites of a decoder layer at Llama-3-8B and
    # Qwen3-14B shapes, batched decode on the down projection, and the mid-size M where HBM-bound turns MMA-bound
    cfgs += [("L3-8B qkv", 2048, 6144, 4096, 2, "normal"), ("L3-8B o-proj", 2048, 4096, 4096, 2, "normal"),
             ("Q3-14B up/gate", 2048, 17408, 5120, 2, "normal"), ("Q3-14B down", 2048, 5120, 17408, 2, "normal"),
             ("Q3-14B qkv", 2048, 7168, 5120, 2, "normal")]
    cfgs += [(f"decode down M={m}", m, 4096, 14336, 2, "normal") for m in (1, 32)]
    cfgs += [(f"decode gate+up M={m}", m, 28672, 4096, 2, "normal") for m in (1, 32)]
    cfgs += [("decode qkv M=1", 1, 6144, 4096, 2, "normal")]
    cfgs += [(f"decode M={m}", m, 4096, 4096, 2, "normal") for m in (64,)]
    cfgs += [(f"mid M={m}", m, 4096, 4096, 2, "normal") for m in (128, 256, 512, 1024)]
    for c in cfgs:
        bench_shape(*c, rows)
    # the paper-faithful scaled residual (HEAL_LO_SCALED, s = 10): two one-product GEMMs summed into one FP32 output
    bench_shape("cfg2 up/gate, s=10 variant", 2048, 14336, 4096, 2, "normal", rows, flags=hb.LO_SCALED)
    bench_shape("cfg1 decode M=8, s=10 variant", 8, 4096, 4096, 2, "normal", rows, flags=hb.LO_SCALED)
    sweep = products_sweep()
    name = torch.cuda.get_device_name(0)
    print(f"# HEAL compensated GEMM on {name}: all BASELINE.json configs\n")
    print(f"Peaks ({src}): cuBLAS BF16 {burst:.0f} TFLOP/s burst / {sust:.0f} sustained; HBM copy {hbm:.0f} GB/s; nominal 2250 TFLOP/s, ~8 TB/s.\n")
    print("Times are medians in microseconds (min in brackets); `full` = heal_gemm (split + GEMM; one fused kernel for M <= 16), "
          "`full + HEAL_B_STATIC` = the same call with the static-weights promise (weights stream before the dependency wait), `G+E` = heal_gemm_presplit "
          "(3P: weights pre-split, the static-weight case).  `tensor` = n_prod x effective rate, as % of measured burst / nominal peak.  "
          "GB/s = (2KN + 4MK + 4MN) / t, as % of the measured copy peak.  cuBLAS columns: torch.matmul on the same inputs "
          "(SGEMM with TF32 off; FP16 and BF16 with operands rounded, 16-bit output).\n")
    print("| config | MxNxK | mode | full us | full + HEAL_B_STATIC us (M <= 64) | G+E us | eff TFLOP/s | tensor TFLOP/s (% burst / % nominal) | GB/s (% peak) | cuBLAS SGEMM us | cuBLAS FP16 us | cuBLAS BF16 us | timing |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    print("\n".join(rows))
    print("\n## What bounds the pair kernel: tensor work per loaded byte (2048x14336x4096, pre-split planes, burst)\n")
    print("The same kernel with 1 / 2 / 3 / 4 products per loaded k-tile (32 / 48 / 64 / 64 KB per CTA and k-tile): the tensor rate rises "
          "with the products per byte until the fourth product makes the tensor pipe the limit, i.e. operand delivery (L2 -> SM), "
          "not the tensor pipe, bounds the 2P kernel (DESIGN.md 7).\n")
    print("| products | us | tensor TFLOP/s | KB per CTA and k-tile | delivery per SM GB/s |")
    print("|---|---|---|---|---|")
    print("\n".join(sweep))


if __name__ == "__main__":
    main()
