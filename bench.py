#!/usr/bin/env python
"""bench.py -- HEAL compensated GEMM on B200: effective TFLOP/s on BASELINE.json configs[2]
(Llama-3-8B-shaped MLP GEMMs, M=2048 prefill tokens, FP32 activations with outlier channels,
FP16 weights, two-product compensation, FP32 output).

One "step" = one pass of the whole hot path (split -> tcgen05 multi-product MMA -> FP32 epilogue)
over one batch of synthetic input, for both MLP GEMMs:
    up/gate : [2048 x 4096]  . [4096 x 14336]
    down    : [2048 x 14336] . [14336 x 4096]
value = sum(2 M N K) / time  (effective TFLOP/s; the tensor cores do n_prod = 2 times that).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--full]

N > 1: one rank per GPU (launched by torchrun; `python bench.py --gpus N` alone re-executes itself under
torch.distributed.run); the path shards over independent token batches (M) with no data-path collective ->
"scaling": "weak".  `--impl reference` times the CPU oracle (as it stands) on a bounded row sample of the same
workload.  Besides the contract keys the line carries the other BASELINE.json configs as context (`small_m`: decode and
LM-head bandwidth, `square`: the three-product sweep, `lm_head_M512`, `cublas_context`, `error_contrast_vs_fp64`,
`elementwise_err_vs_fp64`, `mlp_block`); `--full` adds the qkv / o-proj / Qwen3-14B / mid-size-M table (`shapes`).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "compensated-GEMM effective TFLOP/s (2MNK/time), Llama-3-8B MLP GEMMs, two-product HEAL"
UNIT = "TFLOP/s"
M_TOK, D_MODEL, D_FF = 2048, 4096, 14336
SHAPES = [("up_gate", M_TOK, D_FF, D_MODEL), ("down", M_TOK, D_MODEL, D_FF)]       # (name, M, N, K)
FLOP_STEP = sum(2 * m * n * k for _, m, n, k in SHAPES)
N_PROD = 2
WORKLOAD = ("configs[2]: Llama-3-8B MLP GEMMs, FP32 activations M=2048 x K N(0,1) with x50 outlier channels, "
            "FP16 weights N(0,0.02^2) 4096x14336 (up/gate) and 14336x4096 (down), two-product compensation")


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"burst": d["bf16_tflops"], "sustained": d["bf16_tflops_sustained"], "hbm": d["hbm_gbs"], "src": "measured"}
    return {"burst": 1590.0, "sustained": 1400.0, "hbm": 6650.0, "src": "fallback"}


class ClockSampler(threading.Thread):
    """Samples SM clock, power and clock-event (throttle) reasons through NVML during the timed region."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag, self.err = index, [], False, None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            while not self.stop_flag:
                self.rows.append((float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)),
                                  nv.nvmlDeviceGetPowerUsage(h) / 1000.0,
                                  int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))))
                time.sleep(0.001)
        except Exception as e:  # noqa: BLE001
            self.err = repr(e)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled: %s" % self.err]}
        sm = sorted(r[0] for r in self.rows)
        bits = 0
        for r in self.rows:
            bits |= r[2]
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}
        return {"sm_mhz": sm[len(sm) // 2], "sm_min_mhz": sm[0], "sm_max_mhz": self.max_mhz,
                "reasons": [n for b, n in names.items() if bits & b],
                "power_w_max": max(r[1] for r in self.rows), "samples": len(self.rows)}


def make_inputs(seed, row0=0):
    """The two GEMMs' inputs; `row0` = first row of the global activation matrix this rank owns (rows are regenerable)."""
    from paper_2606_21023_b200 import inputs
    out = []
    for name, M, N, K in SHAPES:
        A = inputs.activations(M, K, seed=seed, outliers=True, row0=row0)
        W = inputs.weights_f16(K, N, seed=seed)
        out.append((name, A, W))
    return out


def oracle_sample(data, rows_per_gemm):
    """Times the CPU oracle (as it stands) on `rows_per_gemm` sampled rows of each GEMM."""
    import oracle
    rows = np.linspace(0, M_TOK - 1, rows_per_gemm).astype(np.int64)
    t0 = time.perf_counter()
    refs = [oracle.gemm_f64(A, W, rows=rows) for _, A, W in data]
    dt = time.perf_counter() - t0
    flop = sum(2 * rows_per_gemm * n * k for _, _, n, k in SHAPES)
    return rows, refs, dt, flop / dt / 1e12, oracle.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    data = make_inputs(0)
    rows_n = 32
    for _ in range(args.warmup):
        oracle_sample(data, 8)
    t = []
    for _ in range(args.steps):
        _, _, dt, tf, cores = oracle_sample(data, rows_n)
        t.append(dt)
    tot = sum(t)
    value = args.steps * sum(2 * rows_n * n * k for _, _, n, k in SHAPES) / tot / 1e12
    sample = f"{rows_n} evenly spaced rows of each of the two GEMMs per step (full N and K)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


L2_BYTES = 126e6


def time_calls(fns, graph, reps=5, cool=0.3):
    """Median microseconds per call of `fns` run back to back (one callable per weight copy) on a side stream: as a
    CUDA graph (launch-latency-scale kernels, rotating over the copies) or as a plain loop; CUDA events on that stream."""
    import torch
    time.sleep(cool)                                    # start from an idle GPU: burst figures
    s = torch.cuda.Stream()
    n_calls = len(fns) if graph else max(len(fns), 10 // len(fns) * len(fns))
    with torch.cuda.stream(s):
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
    return ts[len(ts) // 2]


def shape_report(hb, peaks, M, N, K, nprod, dist="normal", cublas=True, flags=0):
    """One shape through the C ABI: `full` = heal_gemm (FP32 in, everything included), `gemm` = heal_gemm_presplit (steps G + E on
    planes; in 3P the weights are pre-split, the static-weight case), plus cuBLAS SGEMM (TF32 off) / FP16 / BF16 via
    torch.matmul on the same inputs as context.  Inputs are made on the device (timing only; parity lives in tests/)."""
    import torch
    gen = torch.Generator(device="cuda")
    gen.manual_seed(1234)
    w_bytes = K * N * (4 if nprod >= 3 else 2)
    small = 2.0 * nprod * M * N * K < 5e10
    ncopies = max(2, min(12, int(3 * L2_BYTES // w_bytes) + 1)) if small else 1
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
    reps = max(1, 24 // ncopies) if small else 1
    out = {"MxNxK": f"{M}x{N}x{K}", "mode": f"{nprod}P", "timing": f"graph, {ncopies} weight copies" if small else "loop"}
    t_full = time_calls([(lambda b=b: hb.heal_gemm(A, b, nprod | flags, C=C)) for b in Bs] * reps, small)
    ah, al = hb.heal_split(A, lo_shift=hb.LO_SHIFT if flags & hb.LO_SCALED else 0)
    planes = [(hb.heal_split(b) if nprod >= 3 else (b, None)) for b in Bs]
    t_gemm = time_calls([(lambda q=q: hb.heal_gemm_presplit(ah, al, q[0], q[1], nprod | flags, C=C)) for q in planes] * reps, small)
    del planes
    hb.set_workspace(None)
    flop = 2.0 * M * N * K
    byt = K * N * 2 + M * K * 4 + M * N * 4
    out.update({"full_us": t_full, "gemm_us": t_gemm, "eff_tflops_full": flop / t_full / 1e6, "eff_tflops_gemm": flop / t_gemm / 1e6,
                "tensor_tflops_gemm": nprod * flop / t_gemm / 1e6,
                "tensor_frac_of_measured_burst": nprod * flop / t_gemm / 1e6 / peaks["burst"],
                "tensor_frac_of_nominal_2250": nprod * flop / t_gemm / 1e6 / 2250.0})
    if M <= 64:
        out["GBps_full"] = byt / t_full / 1e3
        out["frac_of_measured_hbm_peak"] = byt / t_full / 1e3 / peaks["hbm"]
    if cublas:
        torch.backends.cuda.matmul.allow_tf32 = False
        A16, Ab = A.half(), A.bfloat16()
        C16 = torch.empty(M, N, device="cuda", dtype=torch.float16)
        Cb = torch.empty(M, N, device="cuda", dtype=torch.bfloat16)
        B32 = [b.float() for b in Bs]
        out["cublas_sgemm_us"] = time_calls([(lambda b=b: torch.matmul(A, b, out=C)) for b in B32] * reps, small, reps=3)
        del B32
        B16 = [b.half() for b in Bs]
        out["cublas_fp16_us"] = time_calls([(lambda b=b: torch.matmul(A16, b, out=C16)) for b in B16] * reps, small, reps=3)
        del B16
        Bb = [b.bfloat16() for b in Bs]
        out["cublas_bf16_us"] = time_calls([(lambda b=b: torch.matmul(Ab, b, out=Cb)) for b in Bb] * reps, small, reps=3)
        del Bb
    del Bs
    torch.cuda.empty_cache()
    return out


def mlp_block_report(hb, M=2048):
    """The MLP block of Algorithm 1 at Llama-3-8B size, M tokens, through the fused entry points: Norm -> split,
    gate_up GEMM with the SiLU-mul epilogue (activation planes out), down GEMM adding onto the residual: three launches."""
    import torch
    D, FF = 4096, 14336
    gen = torch.Generator(device="cuda")
    gen.manual_seed(5)
    H = torch.randn(M, D, device="cuda", generator=gen)
    gam = torch.ones(D, device="cuda")
    Wgu = (torch.randn(D, 2 * FF, device="cuda", generator=gen) * 0.02).half()
    Wd = (torch.randn(FF, D, device="cuda", generator=gen) * 0.02).half()
    out = H.clone()
    xh, xl, _ = hb.heal_rmsnorm_split(H, gam)
    _, ah, al = hb.heal_gemm_presplit_ex(xh, xl, Wgu, None, 2 | hb.EPI_SILU_MUL, want_c=False)

    def block():
        hb.heal_rmsnorm_split(H, gam)                                   # (writes fresh planes each call)
        hb.heal_gemm_presplit_ex(xh, xl, Wgu, None, 2 | hb.EPI_SILU_MUL, want_c=False, C_hi=ah, C_lo=al)
        hb.heal_gemm_presplit_ex(ah, al, Wd, None, 2 | hb.EPI_ACCUMULATE, C=out, want_planes=False)

    n0 = hb.launch_count()
    block()
    launches = hb.launch_count() - n0
    t = time_calls([block] * (1 if M > 64 else 8), M <= 64)
    flop = 2.0 * M * D * (2 * FF) + 2.0 * M * FF * D
    byt = 2.0 * (D * 2 * FF + FF * D)                                   # FP16 weights: what a decode-sized block has to stream
    out = {"shape": f"M={M}, d=4096, ff=14336 (gate_up interleaved 4096x28672, down 14336x4096)", "launches": int(launches), "us": t,
           "eff_tflops": flop / t / 1e6, "tensor_tflops": 2 * flop / t / 1e6}
    if M <= 64:
        out["weights_GBps"] = byt / t / 1e3                               # (weights stay the same copy: 352 MB per block > L2)
    return out


def small_m_report(hb, peaks):
    """HBM-bound shapes of BASELINE.json configs[1] (decode 4096x4096, M = 1/8/32) and configs[4] (LM head, M = 1/64), plus the
    down and gate+up projections of a decoder layer at decode batch sizes:
    achieved GB/s = (2KN + 4MK + 4MN) / t through heal_gemm (device buffers; one fused kernel for decode-sized M), timed as a
    CUDA graph of back-to-back calls rotating over enough distinct weight copies to exceed the 126 MB L2; `eager_us` = the
    same calls issued one by one from the host (no graph): host-side launch cost included."""
    import torch
    out = {}
    for tag, M, N, K in [("decode_M1", 1, 4096, 4096), ("decode_M8", 8, 4096, 4096), ("decode_M32", 32, 4096, 4096),
                         ("lm_head_M1", 1, 128256, 4096), ("lm_head_M64", 64, 128256, 4096),
                         # (context beyond BASELINE.json: the two large decode GEMMs of a Llama-3-8B layer)
                         ("layer_down_M8", 8, 4096, 14336), ("layer_gate_up_M1", 1, 28672, 4096)]:
        gen = torch.Generator(device="cuda")
        gen.manual_seed(7)
        ncopies = max(2, min(12, int(3 * L2_BYTES // (K * N * 2)) + 1))
        A = torch.randn(M, K, device="cuda", generator=gen)
        Ws = [(torch.randn(K, N, device="cuda", generator=gen) * 0.02).half() for _ in range(ncopies)]
        C = torch.empty(M, N, device="cuda")
        ws = torch.empty(max(256, hb.workspace_size(M, N, K, hb.MODE_2P)), dtype=torch.uint8, device="cuda")
        hb.set_workspace(ws)
        byt = K * N * 2 + M * K * 4 + M * N * 4
        reps = max(1, 24 // ncopies)
        res = {}
        for name, mode in (("heal_gemm", hb.MODE_2P), ("heal_gemm+B_STATIC", hb.MODE_2P | hb.B_STATIC)):
            fns = [(lambda W=W: hb.heal_gemm(A, W, mode, C=C)) for W in Ws] * reps
            t = time_calls(fns, True, cool=0.5)                    # (idle first: the LM-head shapes are power-sensitive, back-to-back runs drift)
            res[name] = {"us": t, "GB/s": byt / t / 1e3, "frac_of_measured_hbm_peak": byt / t / 1e3 / peaks["hbm"]}
            if name == "heal_gemm":
                res[name]["eager_us"] = time_calls(fns, False, cool=0.5)
                res[name]["kernel"] = hb.last_kernel()
        out[tag] = res
        hb.set_workspace(None)
        del Ws
        torch.cuda.empty_cache()
    return out


def elementwise_stats(X, ref, rows):
    """max / median of |x - ref| / |ref| over the sampled rows (elements with |ref| below 1e-3 of the row's RMS are left
    out of the relative statistics: they are cancellations, where any FP32 algorithm has a large relative error)."""
    d = np.abs(X[rows].astype(np.float64) - ref)
    rms = np.sqrt((ref ** 2).mean(axis=1, keepdims=True))
    keep = np.abs(ref) >= 1e-3 * rms
    rel = d[keep] / np.abs(ref[keep])
    return {"max_rel": float(rel.max()), "median_rel": float(np.median(rel)), "max_abs_over_row_rms": float((d / rms).max())}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_21023_b200 import binding as hb
    from paper_2606_21023_b200 import shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if torch.cuda.device_count() <= local:
        raise SystemExit(f"bench.py: rank {rank} needs cuda:{local}, only {torch.cuda.device_count()} device(s) visible")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hb.lib()

    # M-sharding: the global batch of world x 2048 tokens is cut into contiguous row ranges, one per rank; weights
    # are replicated; no data-path collective.  Rows are regenerable, so rank r generates exactly its rows of the global matrix.
    r0, r1 = shard.shard_rows(world * M_TOK, world, rank)
    assert r1 - r0 == M_TOK
    data = make_inputs(seed=0, row0=r0)
    host = [(n, torch.from_numpy(A).pin_memory(), torch.from_numpy(W).pin_memory()) for n, A, W in data]
    devs = [(n, A.cuda(), W.cuda(), torch.empty((A.shape[0], W.shape[1]), device="cuda")) for n, A, W in host]
    ws = torch.empty(max(hb.workspace_size(m, n, k, hb.MODE_2P) for _, m, n, k in SHAPES), dtype=torch.uint8, device="cuda")
    hb.set_workspace(ws)                                # the timed path never allocates
    stream = torch.cuda.current_stream()

    def step():
        for _, A, W, C in devs:
            hb.heal_gemm(A, W, hb.MODE_2P, C=C)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, n):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(n):
            fn()
        e1.record(stream)
        barrier()
        ms = e0.elapsed_time(e1)
        if world > 1:
            t = torch.tensor([ms], device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms = float(t.item())
        return ms

    for _ in range(max(args.warmup, 3)):
        step()
    sampler = ClockSampler(int(os.environ.get("CUDA_VISIBLE_DEVICES", str(local)).split(",")[local]) if world == 1 else local)
    l0 = hb.launch_count()
    sampler.start()
    time.sleep(0.01)
    ms_total = timed(step, args.steps)
    launches = hb.launch_count() - l0
    ms_step = ms_total / args.steps
    value = shard.aggregate_throughput([FLOP_STEP] * world, [ms_step] * world) / 1e12      # all ranks' flops / the slowest rank's time

    # ---- roofline of the dominant kernel, timed alone on pre-split planes (same launch configuration as in the step)
    planes = []
    for _, A, W, C in devs:
        ah, al = hb.heal_split(A)
        planes.append((ah, al, W, C))

    def gemm_only():
        for ah, al, W, C in planes:
            hb.heal_gemm_presplit(ah, al, W, None, hb.MODE_2P, C=C)

    for _ in range(3):
        gemm_only()
    kernel_name = hb.last_kernel()
    ms_gemm = timed(gemm_only, args.steps) / args.steps / len(SHAPES)        # average launch duration
    sampler.stop_flag = True
    sampler.join()
    peaks = load_peaks()
    long_run = ms_total > 1000.0
    peak = peaks["sustained"] if long_run else peaks["burst"]
    flop_launch = N_PROD * FLOP_STEP / len(SHAPES)
    achieved = flop_launch / (ms_gemm * 1e-3) / 1e12
    traffic, traffic_src = None, None
    tpath = os.path.join(ROOT, "profiles", "gemm_dram_traffic.json")
    if os.path.exists(tpath):
        tj = json.load(open(tpath))
        traffic, traffic_src = tj.get("dram_bytes_per_launch"), tj.get("source")
    # operand delivery (L2 -> SM) of the same launches: the measured limiter of this kernel; per k-tile a CTA
    # receives its 128 rows of A_hi and A_lo and half of the 256-column W tile = 48 KB
    ktile_steps = sum((m // 256) * (n // 256) * (k // 64) for _, m, n, k in SHAPES) * 2 / len(SHAPES)       # CTA k-tile steps per launch
    delivery = 48 * 1024 * ktile_steps / (ms_gemm * 1e-3) / 1e9 / 148

    # ---- end to end through the C ABI with HOST buffers (H2D + path + D2H inside the timed region)
    e2e_steps = max(1, min(args.steps, 5))
    outs = [torch.empty((A.shape[0], W.shape[1]), dtype=torch.float32).pin_memory() for _, A, W in host]

    def step_host():
        for (_, A, W), C in zip(host, outs):
            hb.heal_gemm_host(A, W, hb.MODE_2P, C=C)

    step_host()
    ms_e2e = timed(step_host, e2e_steps) / e2e_steps
    h2d = sum(A.numel() * 4 + W.numel() * 2 for _, A, W in host)
    d2h = sum(C.numel() * 4 for C in outs)

    # ... and the inference form: weights resident on the device, only the step's activations travel in and the results out
    def step_host_act():
        for (_, A, W), (_, _, Wd, _), C in zip(host, devs, outs):
            hb.heal_gemm_host_act(A, Wd, hb.MODE_2P, C=C)

    step_host_act()
    ms_e2e_act = timed(step_host_act, e2e_steps) / e2e_steps
    h2d_act = sum(A.numel() * 4 for _, A, W in host)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f16xf16->f32",
            "data": "synthetic",
            "config": {"workload": WORKLOAD, "global_tokens": world * M_TOK, "parallelism": f"dp{world} over token batches (M-sharding, no collective)",
                       "l2": "inputs larger than L2 (A+W+C = 268 MB per GEMM vs 126 MB L2)",
                       "tensor_tflops": N_PROD * value},
            "roofline": {"bound": "tensor", "kernel": kernel_name, "achieved": achieved, "peak": peak,
                         "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                         "peak_kind": f"{peaks['src']} cuBLAS bf16 {'sustained' if long_run else 'burst'} (fp16 = bf16 rate)",
                         "frac_of_nominal_2250": achieved / 2250.0, "frac_of_measured_burst": achieved / peaks["burst"],
                         "frac_of_measured_sustained": achieved / peaks["sustained"], "avg_launch_ms": ms_gemm,
                         "flops_per_launch": flop_launch,
                         "limiter": {"what": "operand movement per MMA: the SM's shared-memory port (48 KB of TMA writes + 96 KB of tcgen05.mma operand reads per CTA and "
                                             "1024-cycle k-tile) ahead of the L2 -> SM fabric; tensor pipe ~80 % active in ncu",
                                     "achieved_GBps_per_sm": delivery, "probe_peak_GBps_per_sm": 69.4,
                                     "source": "profiles/probes_r01.md, DESIGN.md section 7"}},
            "e2e": {"value": world * FLOP_STEP / (ms_e2e * 1e-3) / 1e12, "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e},
            "e2e_weights_resident": {"value": world * FLOP_STEP / (ms_e2e_act * 1e-3) / 1e12, "unit": UNIT, "h2d_bytes_per_step": h2d_act,
                                     "d2h_bytes_per_step": d2h, "ms_per_step": ms_e2e_act,
                                     "what": "heal_gemm_host_act: FP16 weights stay on the device (the inference case), activations and results cross PCIe every step"},
            "gpu_launches": int(launches),
            "clocks": sampler.summary(),
        }
        if world == 1:
            rows_n = 64
            rows, refs, dt, tf, cores = oracle_sample(data, rows_n)
            line["cpu_baseline"] = {"value": tf, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
                                    "sample": f"{rows_n} evenly spaced rows of each of the two GEMMs (full N and K)"}
            import oracle
            errs, contrast, elem = {}, {}, {}
            torch.backends.cuda.matmul.allow_tf32 = False
            for (name, A, W), (_, Ad, Wd, C), ref in zip(data, devs, refs):
                hb.heal_gemm(Ad, Wd, hb.MODE_2P, C=C)
                heal = C.cpu().numpy()
                fp16 = hb.heal_gemm(Ad, Wd, hb.MODE_1P).cpu().numpy()
                bf16 = torch.matmul(Ad.bfloat16(), Wd.bfloat16()).float().cpu().numpy()
                sgemm = torch.matmul(Ad, Wd.float()).cpu().numpy()
                errs[name] = oracle.normwise_error(heal, ref, A, W, rows=rows)
                # context (north_star): the same inputs through plain 16-bit GEMMs and cuBLAS SGEMM, scored the same way
                e = lambda X: oracle.normwise_error(X, ref, A, W, rows=rows)
                contrast[name] = {"heal_2P": errs[name], "plain_fp16_1P (heal_gemm mode 1)": e(fp16),
                                  "plain_bf16 (cuBLAS, bf16 out)": e(bf16), "sgemm_fp32 (cuBLAS, TF32 off)": e(sgemm)}
                # element-wise view of "near-FP32": relative error per element on the sampled rows
                elem[name] = {"heal_2P": elementwise_stats(heal, ref, rows), "sgemm_fp32 (cuBLAS, TF32 off)": elementwise_stats(sgemm, ref, rows),
                              "plain_fp16_1P": elementwise_stats(fp16, ref, rows)}
            line["normwise_err_vs_fp64"] = errs
            line["error_contrast_vs_fp64"] = contrast
            line["elementwise_err_vs_fp64"] = elem
            del devs, planes
            torch.cuda.empty_cache()
            # ---- the other BASELINE.json configs and context rows (CUDA-event timings of the same process, burst regime)
            line["cublas_context"] = {name: {k: v for k, v in shape_report(hb, peaks, m, n, k_, 2).items() if k.startswith("cublas") or k in ("full_us", "gemm_us")}
                                      for name, m, n, k_ in SHAPES}
            line["small_m"] = small_m_report(hb, peaks)
            line["square"] = {str(n): shape_report(hb, peaks, n, n, n, 3, dist="uniform") for n in (1024, 2048, 4096, 8192)}
            line["lm_head_M512"] = shape_report(hb, peaks, 512, 128256, 4096, 2)
            line["mlp_block"] = mlp_block_report(hb)
            line["mlp_block_decode_M8"] = mlp_block_report(hb, M=8)
            if args.full:
                extra = [("L3-8B qkv", 2048, 6144, 4096), ("L3-8B o-proj", 2048, 4096, 4096), ("Q3-14B gate_up", 2048, 17408, 5120),
                         ("Q3-14B down", 2048, 5120, 17408), ("Q3-14B qkv", 2048, 7168, 5120), ("decode down M=1", 1, 4096, 14336),
                         ("decode down M=32", 32, 4096, 14336), ("decode gate+up M=1", 1, 28672, 4096), ("decode qkv M=1", 1, 6144, 4096),
                         ("decode M=64", 64, 4096, 4096), ("mid M=128", 128, 4096, 4096), ("mid M=256", 256, 4096, 4096),
                         ("mid M=512", 512, 4096, 4096), ("mid M=1024", 1024, 4096, 4096), ("cfg0 single (3P)", 64, 256, 256)]
                line["shapes"] = {name: shape_report(hb, peaks, m, n, k_, 3 if "3P" in name else 2) for name, m, n, k_ in extra}
                line["shapes"]["cfg2 up/gate, s=10 (HEAL_LO_SCALED)"] = shape_report(hb, peaks, 2048, 14336, 4096, 2, cublas=False, flags=hb.LO_SCALED)
                line["shapes"]["decode M=8, s=10 (HEAL_LO_SCALED)"] = shape_report(hb, peaks, 8, 4096, 4096, 2, cublas=False, flags=hb.LO_SCALED)
                line["shapes"]["cfg2 up/gate, HEAL_FUSE_SPLIT"] = shape_report(hb, peaks, 2048, 14336, 4096, 2, cublas=False, flags=hb.FUSE_SPLIT)
        print(json.dumps(line))
    hb.set_workspace(None)
    if world > 1:
        dist.destroy_process_group()


def run_trace():
    """`bench.py --trace`: builds libheal_trace.so (the same sources with -DHEAL_TRACE) and prints, as markdown, (1) the %globaltimer
    phase stamps of the decode GEMM 4096 x 4096 (M = 1, 32) inside a CUDA graph of twelve launches rotating over twelve weight copies,
    (2) the same graph with ONE weight copy (weights resident in L2: the latency floor of the kernel structure), (3) the wait counters of
    the CTA-pair kernel on the two MLP GEMMs.  Diagnostics only: nothing here is a bench value."""
    import ctypes
    import torch
    from paper_2606_21023_b200 import build as hbuild
    from paper_2606_21023_b200 import binding as hb
    hb.LIB_PATH = hbuild.build(trace=True)
    L = hb.lib()
    L.heal_debug_set_trace.argtypes = [ctypes.c_void_p]
    names = {0: "kernel entry", 13: "TMEM allocated", 1: "prologue done", 2: "griddepcontrol.wait returned", 3: "first TMA issued",
             4: "first operand tile complete", 5: "last MMA issued", 6: "commit seen by epilogue", 7: "partials pushed",
             8: "all partials landed (owners)", 9: "C stored", 11: "TMEM released"}
    print("# Phase trace of the small-M kernel and wait counters of the CTA-pair kernel (`python bench.py --trace`, trace build)\n")
    for M in (1, 32):
        for ncopies in (12, 1):
            gen = torch.Generator(device="cuda")
            gen.manual_seed(7)
            A = torch.randn(M, 4096, device="cuda", generator=gen)
            Ws = [(torch.randn(4096, 4096, device="cuda", generator=gen) * 0.02).half() for _ in range(ncopies)]
            C = torch.empty(M, 4096, device="cuda")
            tr = torch.zeros(16 * 1024 * 64, dtype=torch.int64, device="cuda")
            s = torch.cuda.Stream()
            with torch.cuda.stream(s):
                for W in Ws:
                    hb.heal_gemm(A, W, hb.MODE_2P, C=C)
                s.synchronize()
                L.heal_debug_set_trace(ctypes.c_void_p(tr.data_ptr()))
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=s):
                    for i in range(12):
                        hb.heal_gemm(A, Ws[i % ncopies], hb.MODE_2P, C=C)
                for _ in range(3):
                    g.replay()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(s)
                g.replay()
                e1.record(s)
                s.synchronize()
            L.heal_debug_set_trace(None)
            t = tr.cpu().numpy().reshape(16, 1024, 64)
            a, nxt = t[6], t[7]
            act = a[:, 0] > 0
            base = a[act, 2].min()
            print(f"## decode {M} x 4096 x 4096, {hb.last_kernel()}, {int(act.sum())} CTAs, {ncopies} weight cop{'y (L2-resident)' if ncopies == 1 else 'ies (HBM)'}: "
                  f"{e0.elapsed_time(e1) * 1e3 / 12:.2f} us per GEMM in the graph\n")
            print("| phase (us after the launch's earliest griddepcontrol.wait return) | min | median | max |\n|---|---|---|---|")
            for k in (0, 13, 1, 2, 3, 4, 5, 6, 7, 8, 9, 11):
                v = a[act, k]
                v = v[v > 0]
                if v.size:
                    print(f"| {names[k]} | {(v.min() - base) / 1e3:.2f} | {(np.median(v) - base) / 1e3:.2f} | {(v.max() - base) / 1e3:.2f} |")
            print(f"| next launch: griddepcontrol.wait returned | {(nxt[nxt[:, 0] > 0, 2].min() - base) / 1e3:.2f} | | |\n")
    L.heal_debug_read_pair_trace.argtypes = [ctypes.c_void_p, ctypes.c_int]
    print("## CTA-pair kernel: where the MMA thread and an epilogue warp wait (clock64 counters, median over the 74 pairs)\n")
    print("| GEMM | MMA thread: waits for operands | waits for a free accumulator | issues | epilogue warp: waits for a segment | drains TMEM (cycles per segment) | stores C (cycles per tile) |\n|---|---|---|---|---|---|---|")
    for name, M, N, K in SHAPES:
        A = torch.randn(M, K, device="cuda")
        W = (torch.randn(K, N, device="cuda") * 0.02).half()
        ah, al = hb.heal_split(A)
        C = torch.empty(M, N, device="cuda")
        for _ in range(5):
            hb.heal_gemm_presplit(ah, al, W, None, hb.MODE_2P, C=C)
        torch.cuda.synchronize()
        buf = (ctypes.c_ulonglong * (74 * 8))()
        L.heal_debug_read_pair_trace(buf, 74 * 8)
        t = np.array(buf[:], dtype=np.float64).reshape(74, 8)
        tiles = (M // 256) * (N // 256) / 74.0
        print(f"| {name} {M}x{N}x{K} | {np.median(t[:, 0] / t[:, 2]) * 100:.1f} % | {np.median(t[:, 1] / t[:, 2]) * 100:.1f} % | "
              f"{100 - np.median((t[:, 0] + t[:, 1]) / t[:, 2]) * 100:.1f} % | {np.median(t[:, 3] / t[:, 6]) * 100:.1f} % | "
              f"{np.median(t[:, 4] / t[:, 6]) * 100:.1f} % ({np.median(t[:, 4] / t[:, 7]):.0f}) | {np.median(t[:, 5] / t[:, 6]) * 100:.1f} % ({np.median(t[:, 5]) / tiles:.0f}) |")


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` (N > 1) outside torchrun: start N ranks of this script, one per GPU, rendezvous on 127.0.0.1."""
    import subprocess
    import torch
    if not torch.cuda.is_available() or torch.cuda.device_count() < args.gpus:
        n = torch.cuda.device_count() if torch.cuda.is_available() else 0
        raise SystemExit(f"bench.py: --gpus {args.gpus} needs {args.gpus} CUDA devices, {n} visible")
    port = 29500 + os.getpid() % 1000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__), "--gpus", str(args.gpus), "--steps", str(args.steps),
           "--warmup", str(args.warmup), "--impl", args.impl] + (["--full"] if args.full else [])
    raise SystemExit(subprocess.call(cmd))


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1500)      # > 1 s of back-to-back GEMMs: the sustained (power-capped) regime
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--full", action="store_true", help="also time the qkv / o-proj / Qwen3-14B / mid-size-M shapes (key `shapes`)")
    ap.add_argument("--trace", action="store_true", help="diagnostics: phase stamps / wait counters from a -DHEAL_TRACE build (markdown)")
    a = ap.parse_args()
    if a.trace:
        run_trace()
        raise SystemExit(0)
    if a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_under_torchrun(a)
    run_reference(a) if a.impl == "reference" else run_ours(a)
