#!/usr/bin/env python
"""bench.py -- W4A4G4 triple-branch linear, fwd + bwd, on synthetic FLUX.1-dev-shaped input.

A step = one pass of the whole hot path (rows a0-a5) over one batch:
    ft_linear_fwd (one kernel: tensor amax + quantize + down-projection of X; its slot sums; 4-bit GEMM + up-projection)
    ft_linear_bwd (dB^T partials with the amax of G as a by-product; quantize + down-projection of G; slot sums of P and
                   dB^T; 4-bit GEMM with Q(R)^T; dA)                                       -- 8 kernel launches
Workload at N=1: BASELINE.json configs[1] (C2): fused QKV projection M=4608, K=3072, N=9216,
stabilizer rank 32, LoRA rank 32.  N>1: every rank runs the same layer on its own batch of 4608
tokens (weak scaling) and all-reduces the LoRA gradients (NCCL), the path's only exchange.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
prints ONE JSON line (rank 0).  --impl reference times the CPU oracle on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

WORKLOAD = dict(name="C2 FLUX.1-dev fused QKV projection", M=4608, K=3072, N=9216, r_s=32, r=32, seed=1)
METRIC = "W4A4G4 linear fwd+bwd TFLOPS (4*M*N*K per step / step time)"
UNIT = "TFLOP/s"
FP4_OVER_BF16 = 4.0   # nominal dense ratio 9 / 2.25 PFLOP/s (B200_PROFILING.md)
FP4_NOMINAL_TFLOPS = 9000.0   # dense NVFP4, B200 (B200_PROFILING.md): the peak north_star's 60 % bar refers to
# dram__bytes_read.sum + dram__bytes_write.sum per launch (bytes) from the ncu --set full capture of the C2 step
# summarised in profiles/r02_full_summary.md (ncu flushes the caches before every launch: cold-cache figures; the
# quantize entries include their k_finalize_h launch)
NCU_DRAM_TRAFFIC = {"gemm_fwd": 62.30e6, "gemm_dgrad": 45.00e6, "quantize_X": 34.67e6, "quantize_G": 102.86e6,
                    "wgrad_dBt": 89.46e6, "wgrad_dA": 29.31e6}
PROBE_SRC = os.path.join(ROOT, "bench_fp4_probe.cu")
PROBE_BIN = os.path.join(ROOT, "build", "bench_fp4_probe")


def build_fp4_probe():
    """nvcc the FP4 tensor-core probe (bench_fp4_probe.cu) into build/ if it is missing or stale."""
    if os.path.exists(PROBE_BIN) and os.path.getmtime(PROBE_BIN) >= os.path.getmtime(PROBE_SRC):
        return PROBE_BIN
    os.makedirs(os.path.dirname(PROBE_BIN), exist_ok=True)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "--expt-relaxed-constexpr",
                    "-I", ROOT, "-o", PROBE_BIN, PROBE_SRC, "-lcuda"], check=True, capture_output=True)
    return PROBE_BIN


def run_fp4_probe(seconds, gpu_index):
    """MMA-only FP4 rate (operands resident in shared memory, no TMA, no epilogue) sustained for `seconds`,
    with the SM clock sampled meanwhile: the measured ceiling next to the nominal 9 PFLOP/s."""
    try:
        exe = build_fp4_probe()
        sampler = ClockSampler(gpu_index)
        sampler.start()
        env = dict(os.environ, CUDA_VISIBLE_DEVICES=os.environ.get("CUDA_VISIBLE_DEVICES", str(gpu_index)))
        r = subprocess.run([exe, "--sustained", str(seconds)], capture_output=True, text=True, timeout=120, env=env)
        clocks = sampler.stop()
        line = [l for l in r.stdout.splitlines() if l.startswith("sustained")]
        if r.returncode != 0 or not line:
            return {"error": (r.stdout + r.stderr)[-300:]}
        tf = float(line[0].split()[-2])
        cyc = float(line[0].split("launches:")[1].split()[0])
        return {"tflops": tf, "cycles_per_mma_m256_n256_k64": cyc, "seconds": seconds, "sm_mhz_median": clocks["sm_mhz"],
                "reasons": clocks["reasons"], "raw": line[0]}
    except Exception as e:   # noqa: BLE001
        return {"error": str(e)[-300:]}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sustained=d.get("bf16_tflops_sustained"),
                    source="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = sorted(int(r[0]) for r in self.rows if r and r[0].isdigit())
        mx = [int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 2 + i and r[2 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# ------------------------------------------------------------------ CPU oracle arm
def oracle_sample(rows=256, repeats=1):
    """The oracle as it stands on a bounded sample of the workload: the first `rows` tokens of
    the C2 batch through forward + dgrad + wgrad against the full-size weight.  Offline parts
    (Eq. 1 split, Q(R)) are outside the timed region, as on the GPU."""
    import numpy as np
    from oracle import layer as olayer
    from oracle import nvfp4
    from paper_2607_05711_b200 import synth
    w = WORKLOAD
    rng = synth.make_rng(w["seed"])
    X = synth.outlier_normal(rng, rows, w["K"])
    R = synth.normal(rng, (w["N"], w["K"]), 0.02)
    r_t = w["r_s"] + w["r"]
    D_f = synth.normal(rng, (w["K"], r_t), 0.01)
    U_f = synth.normal(rng, (r_t, w["N"]), 0.01)
    G = synth.student_t_grad(rng, rows, w["N"])
    qR = olayer.quantize_weight(R)
    times = []
    for _ in range(repeats):
        t0 = time.perf_counter()
        f = olayer.forward(X, qR, D_f, U_f, prescale=True)
        b = olayer.dgrad(G, qR, D_f, U_f, prescale=True)
        olayer.wgrad(X, G, f["H"], b["P"], w["r_s"])
        times.append(time.perf_counter() - t0)
    flops = 4.0 * rows * w["N"] * w["K"]
    return flops, times


def cpu_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    rows = WORKLOAD["M"]
    oracle_sample(rows, 1)                                   # warm-up (BLAS threads, page faults)
    steps = max(1, min(args.steps, 4))                       # each step ~5 s of CPU work
    flops, times = oracle_sample(rows, steps)
    t = sum(times) / len(times)
    val = flops / t / 1e12
    sample = "all %d tokens of C2 (M=%d), fwd+dgrad+wgrad, %d step(s)" % (rows, WORKLOAD["M"], steps)
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
           "warmup": 1, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": WORKLOAD["name"], **{k: WORKLOAD[k] for k in ("M", "K", "N", "r_s", "r")},
                      "sample_rows": rows},
           "cpu_baseline": {"value": val, "unit": UNIT, "cores": cpu_cores(), "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


# ------------------------------------------------------------------ GPU arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2607_05711_b200 import binding as B
    from paper_2607_05711_b200 import build as _build
    from paper_2607_05711_b200 import parallel, prepare

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    _build.build()
    B.lib()                                   # fails loudly if the CUDA library is missing
    w = WORKLOAD
    M, K, N, r_s, r = w["M"], w["K"], w["N"], w["r_s"], w["r"]
    r_t = r_s + r
    peaks = load_peaks()

    # ---- synthetic inputs, generated on the host (seeded), resident in HBM before timing
    import numpy as np
    from paper_2607_05711_b200 import synth
    rng = synth.make_rng(w["seed"] + 1000 * rank)
    Xh = torch.from_numpy(synth.outlier_normal(rng, M, K)).to(torch.bfloat16).pin_memory()
    Wt = torch.from_numpy(synth.normal(rng, (N, K), 0.02)).to(torch.bfloat16).to(dev)
    A = torch.from_numpy(synth.normal(rng, (K, r), 0.01)).to(torch.bfloat16).to(dev)
    Bt = torch.from_numpy(synth.normal(rng, (N, r), 0.01)).to(torch.bfloat16).to(dev)
    Gh = torch.from_numpy(synth.student_t_grad(rng, M, N)).to(torch.bfloat16).pin_memory()
    R, L1, L2t = prepare.random_range_split(Wt, r_s, seed=w["seed"])     # offline (Eq. 1)
    D_f = torch.cat([L1, A], 1).contiguous()
    U_t = torch.cat([L2t, Bt], 1).contiguous()
    layer = B.Layer(R, D_f, U_t, r_s, r, tokens=M)                       # offline: Q(R), both packings; tile-cut scales for M tokens
    X, G = Xh.to(dev), Gh.to(dev)
    y = torch.empty(M, N, dtype=torch.bfloat16, device=dev)
    dx = torch.empty(M, K, dtype=torch.bfloat16, device=dev)
    h = torch.empty(M, r_t, dtype=torch.bfloat16, device=dev)
    p = torch.empty(M, r_t, dtype=torch.bfloat16, device=dev)
    ws = B.new_workspace(M, max(K, N), max(K, N), r_t, dev)
    qx, qg = B.QTensor(M, K, device=dev), B.QTensor(M, N, device=dev)
    dA = torch.empty(K, r, dtype=torch.float32, device=dev)
    dBt = torch.empty(N, r, dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream()

    def step():
        B.ft_linear_fwd(layer, X, y, h, qx, ws)
        B.ft_linear_bwd(layer, X, G, h, dx, p, dA, dBt, qg, ws)
        if world > 1:
            parallel.allreduce_lora_grads(dA, dBt)
    # fwd: k_quantize_fused (single pass, amax inside) + k_finalize_h + k_gemm4_pair; bwd (ft_linear_bwd): k_wgrad
    # (dB^T + amax of G) + k_quantize_fused (streaming) + k_finalize_h + k_gemm4_pair + k_wgrad (dA): 8 kernels, no clear
    # kernel and no memset node (the workspace's control words are put back by the kernels that use them)
    KERNELS_PER_STEP = 8

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    # the launch-bound prologue (amax, quantize) is short: replay the step as a CUDA graph at
    # N=1 so the host never gates the device; eager otherwise
    graph, launch = None, "eager"
    if world == 1 and not args.eager:
        try:
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g):
                step()
            g.replay()
            torch.cuda.synchronize()
            graph, launch = g, "cuda_graph"
        except Exception as e:   # noqa: BLE001
            sys.stderr.write("graph capture failed (%s): eager launches\n" % e)
            torch.cuda.synchronize()
    run = (graph.replay if graph is not None else step)
    for _ in range(3):
        run()
    barrier()

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        run()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    tmax = torch.tensor([ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    ms_per_step = float(tmax.item()) / args.steps
    flops_step = 4.0 * M * N * K
    value = world * flops_step / (ms_per_step * 1e-3) / 1e12

    # ---- end to end through the public API with HOST buffers: H2D of X and G, D2H of every result
    yh = torch.empty(M, N, dtype=torch.bfloat16).pin_memory()
    dxh = torch.empty(M, K, dtype=torch.bfloat16).pin_memory()
    dAh = torch.empty(K, r, dtype=torch.float32).pin_memory()
    dBh = torch.empty(N, r, dtype=torch.float32).pin_memory()

    # Every step copies its inputs from pinned host memory and its results back; the three legs run on
    # three streams with double-buffered device tensors, so the H2D of step i+1 and the D2H of step i-1
    # overlap the kernels of step i (PCIe is full duplex).  The timed region still contains every copy.
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    Xd, Gd = [X, torch.empty_like(X)], [G, torch.empty_like(G)]
    yd, dxd = [y, torch.empty_like(y)], [dx, torch.empty_like(dx)]
    dAd, dBd = [dA, torch.empty_like(dA)], [dBt, torch.empty_like(dBt)]
    ev_in = [torch.cuda.Event() for _ in range(2)]      # inputs of buffer b are on the device
    ev_comp = [torch.cuda.Event() for _ in range(2)]    # kernels of buffer b are done
    ev_out = [torch.cuda.Event() for _ in range(2)]     # results of buffer b are on the host
    for b in range(2):
        ev_comp[b].record(stream)
        ev_out[b].record(stream)

    def e2e_step(i):
        b = i & 1
        with torch.cuda.stream(s_in):
            s_in.wait_event(ev_comp[b])                 # the kernels that last read this buffer are done
            Xd[b].copy_(Xh, non_blocking=True)
            Gd[b].copy_(Gh, non_blocking=True)
            ev_in[b].record(s_in)
        stream.wait_event(ev_in[b])
        stream.wait_event(ev_out[b])                    # the previous results in this buffer have left
        B.ft_linear_fwd(layer, Xd[b], yd[b], h, qx, ws)
        B.ft_linear_bwd(layer, Xd[b], Gd[b], h, dxd[b], p, dAd[b], dBd[b], qg, ws)
        if world > 1:
            parallel.allreduce_lora_grads(dAd[b], dBd[b])
        ev_comp[b].record(stream)
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_comp[b])
            yh.copy_(yd[b], non_blocking=True)
            dxh.copy_(dxd[b], non_blocking=True)
            dAh.copy_(dAd[b], non_blocking=True)
            dBh.copy_(dBd[b], non_blocking=True)
            ev_out[b].record(s_out)

    def e2e_drain():
        stream.wait_stream(s_in)
        stream.wait_stream(s_out)
    e2e_step(0)
    e2e_step(1)
    e2e_drain()
    barrier()
    n_e2e = max(4, min(args.steps, 20))
    e0.record()
    for i in range(n_e2e):
        e2e_step(i)
    e2e_drain()                                         # the last results are on the host inside the timed region
    e1.record()
    barrier()
    te = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
    e2e_ms = float(te.item()) / n_e2e
    clocks = sampler.stop()
    h2d = (Xh.numel() + Gh.numel()) * 2
    d2h = (yh.numel() + dxh.numel()) * 2 + (dAh.numel() + dBh.numel()) * 4

    # ---- per-kernel breakdown.  Each call is captured N times back to back in ONE CUDA graph, cycling over
    # enough copies of its input that the copies together exceed twice the L2 (so every launch reads its tensor from
    # HBM, as in a training step), and the graph is replayed: kernel-to-kernel time, no launch gap, no L2 flush in
    # the timed region.  The GEMMs replay on the same operands (42 MB: L2-resident in the real step as well).
    hs = B.workspace_hs(ws, M, r_t)
    amax = torch.empty(1, dtype=torch.float32, device=dev)

    def graph_us(fns, n=20):
        for f in fns:
            f()
        torch.cuda.synchronize()
        gg = torch.cuda.CUDAGraph()
        with torch.cuda.graph(gg):
            for f in fns:
                f()
        for _ in range(3):
            gg.replay()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(n):
            gg.replay()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / (n * len(fns)) * 1e3

    def copies(t, total_bytes=300e6):
        k = max(2, int(total_bytes // (t.numel() * t.element_size())) + 1)
        return [t] + [t.clone() for _ in range(k - 1)]

    Xs, Gs = copies(X), copies(G)
    kern = {}
    kern["amax_X_us"] = graph_us([lambda x=x: B.ft_tensor_amax(x, amax) for x in Xs])
    kern["quantize_X_a0a1_us"] = graph_us([lambda x=x: B.ft_quantize_blockwise(
        x, qx, down=D_f, h_out=h, hs_out=hs, other_dec_scale=layer.r_kmajor.tensor_dec_scale, workspace=ws) for x in Xs])
    amax_g = B.ft_tensor_amax(G)
    kern["amax_G_us"] = graph_us([lambda g_=g_: B.ft_tensor_amax(g_, amax) for g_ in Gs])
    kern["quantize_G_a3_us"] = graph_us([lambda g_=g_: B.ft_quantize_blockwise(
        g_, qg, tensor_amax=amax_g, down=U_t, h_out=p, hs_out=hs, other_dec_scale=layer.r_nmajor.tensor_dec_scale,
        workspace=ws) for g_ in Gs])
    B.ft_quantize_blockwise(X, qx, down=D_f, h_out=h, hs_out=hs, other_dec_scale=layer.r_kmajor.tensor_dec_scale,
                            workspace=ws)
    kern["gemm_fwd_us"] = graph_us([lambda: B.ft_gemm4(qx, layer.r_kmajor, hs, U_t, y)] * 4)
    B.ft_quantize_blockwise(G, qg, tensor_amax=amax_g, down=U_t, h_out=p, hs_out=hs,
                            other_dec_scale=layer.r_nmajor.tensor_dec_scale, workspace=ws)
    kern["gemm_dgrad_us"] = graph_us([lambda: B.ft_gemm4(qg, layer.r_nmajor, hs, D_f, dx)] * 4)
    kern["wgrad_dA_dBt_us"] = graph_us([lambda g_=g_, x=Xs[i % len(Xs)]: B.ft_lora_wgrad(layer, x, g_, h, p, dA, dBt)
                                        for i, g_ in enumerate(Gs)])
    kern["wgrad_saved4_us"] = graph_us([lambda g_=g_: B.ft_lora_wgrad_q4(layer, qx, g_, h, p, dA, dBt) for g_ in Gs])
    kern["fwd_us"] = graph_us([lambda x=x: B.ft_linear_fwd(layer, x, y, h, qx, ws) for x in Xs])
    kern["bwd_us"] = graph_us([lambda g_=g_, x=Xs[i % len(Xs)]: B.ft_linear_bwd(layer, x, g_, h, dx, p, dA, dBt, qg, ws)
                               for i, g_ in enumerate(Gs)])

    # the same step with 4-bit saved activations (NEXT-2): fwd + ft_linear_bwd_q4, as a CUDA graph
    def step_saved4():
        B.ft_linear_fwd(layer, X, y, h, qx, ws)
        B.ft_linear_bwd_q4(layer, qx, G, h, dx, p, dA, dBt, qg, ws)

    def step_bf16x():
        B.ft_linear_fwd(layer, X, y, h, qx, ws)
        B.ft_linear_bwd(layer, X, G, h, dx, p, dA, dBt, qg, ws)
    kern["step_saved4_us"] = graph_us([step_saved4], 100)
    kern["step_bf16x_us"] = graph_us([step_bf16x], 100)

    # single-copy weights (NEXT-5): the codes of Q(R)^T are rebuilt into a scratch buffer before every backward
    codes_nmajor = layer.r_nmajor.codes
    scratch_t = torch.empty_like(codes_nmajor)

    def step_single_copy():
        B.ft_linear_fwd(layer, X, y, h, qx, ws)
        B.ft_weight_transpose_codes(layer, scratch_t)
        B.ft_linear_bwd(layer, X, G, h, dx, p, dA, dBt, qg, ws)
    layer.r_nmajor.codes = scratch_t
    kern["step_single_copy_us"] = graph_us([step_single_copy], 100)
    layer.r_nmajor.codes = codes_nmajor
    # the transposition alone, over enough distinct destinations that none of it stays in L2
    scr = copies(scratch_t)
    kern["transpose_codes_us"] = graph_us([lambda d=d: B.ft_weight_transpose_codes(layer, d) for d in scr])
    del scr

    # the step WITHOUT a graph: 8 launches enqueued by the host each step (tensor maps come from the library's memo)
    def eager_us(fn, n=50):
        for _ in range(5):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(n):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / n * 1e3
    kern["step_eager_us"] = eager_us(step_bf16x)
    del Xs, Gs
    torch.cuda.empty_cache()

    # bf16 cuBLAS LoRA layer on the same GPU, same shapes, same protocol (CUDA graph, back-to-back replays)
    Am, Bm = A, Bt.t().contiguous()

    def bf16_lora():
        xa = X @ Am
        yy = X @ Wt.t() + xa @ Bm                     # noqa: F841
        gb = G @ Bm.t()
        dxx = G @ Wt + gb @ Am.t()                    # noqa: F841
        da = X.t() @ gb                               # noqa: F841
        db = xa.t() @ G                               # noqa: F841
    bf16_us = graph_us([bf16_lora], 20)

    extra = {}
    if rank == 0 and world == 1 and not args.no_sweep:
        del yh, dxh
        extra = sweep(B, prepare, dev, graph_us, peaks, full=not args.c4_only)
    probe = run_fp4_probe(args.probe_seconds, local) if (rank == 0 and args.probe_seconds > 0) else None
    out = None
    if rank == 0:
        fp4_derived = peaks["bf16"] * FP4_OVER_BF16
        fp4_probe = probe["tflops"] if probe and "tflops" in probe else None
        gemm_flop = 2.0 * M * N * K

        def gemm_entry(name, us, step):
            tf = gemm_flop / (us * 1e-6) / 1e12
            return {"kernel": "k_gemm4_pair (%s)" % name, "step": step, "bound": "tensor", "work": gemm_flop, "work_unit": "flop",
                    "us": round(us, 2), "achieved": tf, "unit": "TFLOP/s", "peak": FP4_NOMINAL_TFLOPS, "frac": tf / FP4_NOMINAL_TFLOPS,
                    "frac_of_probe": (tf / fp4_probe) if fp4_probe else None, "frac_of_derived": tf / fp4_derived,
                    "traffic": NCU_DRAM_TRAFFIC["gemm_" + name]}

        def hbm_entry(kernel, step, nbytes, us, key):
            gbs = nbytes / us / 1e3
            return {"kernel": kernel, "step": step, "bound": "hbm", "work": nbytes, "work_unit": "bytes", "us": round(us, 2),
                    "achieved": gbs, "unit": "GB/s", "peak": peaks["hbm"], "frac": gbs / peaks["hbm"],
                    "frac_of_nominal_8TBps": gbs / 8000.0,
                    "traffic": None if key is None else (NCU_DRAM_TRAFFIC["wgrad_dBt"] + NCU_DRAM_TRAFFIC["wgrad_dA"]
                                                         if key == "wgrad_step" else NCU_DRAM_TRAFFIC[key])}
        qb = 2.5625 + 4.0 * r_t / K                       # codes + scales + H, Hs and the D slice per element of X
        qbg = 2.5625 + 4.0 * r_t / N
        roofs = [
            gemm_entry("fwd", kern["gemm_fwd_us"], "a2"),
            gemm_entry("dgrad", kern["gemm_dgrad_us"], "a4"),
            hbm_entry("k_quantize_fused<64,single> + k_finalize_h (X: amax + quantize + projection, one call)", "a0+a1",
                      qb * M * K, kern["quantize_X_a0a1_us"], "quantize_X"),
            hbm_entry("k_quantize_fused<64,streaming> + k_finalize_h (G, amax given)", "a3", qbg * M * N,
                      kern["quantize_G_a3_us"], "quantize_G"),
            hbm_entry("ft_lora_wgrad: k_wgrad<32,256> (dA and dB^T in one launch of cluster CTAs: reads X and G once)",
                      "a5", 2.0 * M * (K + N), kern["wgrad_dA_dBt_us"], None),
            hbm_entry("k_wgrad_s<32> dB^T (+ amax of G, clears dA) and dA inside ft_linear_bwd: bwd_us - a3 - a4 (derived: "
                      "the dA launch runs partly beside the dgrad GEMM's tail)", "a5 in the step", 2.0 * M * (K + N),
                      kern["bwd_us"] - kern["quantize_G_a3_us"] - kern["gemm_dgrad_us"], "wgrad_step"),
        ]
        gemm_us = 0.5 * (kern["gemm_fwd_us"] + kern["gemm_dgrad_us"])
        gemm_tflops = gemm_flop / (gemm_us * 1e-6) / 1e12
        cpu_flops, cpu_times = oracle_sample(M, 2)
        cpu_val = cpu_flops / (sum(cpu_times) / 2) / 1e12
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "nvfp4 (e2m1 x ue4m3, fp32 accumulate) + bf16 low-rank", "data": "synthetic",
            "config": {"workload": w["name"], "M": M, "K": K, "N": N, "r_s": r_s, "r": r, "tokens_per_gpu": M,
                       "launch": launch, "l2": "step working set ~330 MB > 126 MB L2; per-kernel timings cycle over input "
                                                "copies that together exceed 2 x L2",
                       "parallelism": "dp%d (tokens), all-reduce of dA,dB only" % world,
                       "peaks": peaks["source"]},
            "clocks": clocks,
            "e2e": {"value": world * flops_step / (e2e_ms * 1e-3) / 1e12, "unit": UNIT, "ms_per_step": e2e_ms,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "how": "ft_linear_fwd + ft_linear_bwd per step with X, G copied from pinned host memory and Y, dX, dA, "
                           "dB^T copied back every step; copies on two side streams with double-buffered device tensors "
                           "(H2D of step i+1 and D2H of step i-1 overlap the kernels of step i); PCIe-bound"},
            "gpu_launches": KERNELS_PER_STEP * args.steps,
            "roofline": {"kernel": "k_gemm4_pair (mean of the forward and the dgrad launch: the dominant kernel, %.0f %% of "
                                   "the step)" % (100.0 * (kern["gemm_fwd_us"] + kern["gemm_dgrad_us"]) / (ms_per_step * 1e3)),
                         "bound": "tensor", "achieved": gemm_tflops, "peak": FP4_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                         "frac": gemm_tflops / FP4_NOMINAL_TFLOPS,
                         "peak_note": "nominal dense NVFP4 peak of B200 (B200_PROFILING.md); MEASURED_PEAKS.json holds no FP4 "
                                      "figure, so two measured ceilings are reported beside it",
                         "frac_of_probe": (gemm_tflops / fp4_probe) if fp4_probe else None,
                         "frac_of_derived": gemm_tflops / fp4_derived,
                         "derived_peak": fp4_derived,
                         "derived_note": "measured bf16 burst %.1f x nominal fp4/bf16 ratio 4 (of %s)" % (peaks["bf16"], peaks["source"]),
                         "traffic": 0.5 * (NCU_DRAM_TRAFFIC["gemm_fwd"] + NCU_DRAM_TRAFFIC["gemm_dgrad"])},
            "roofline_kernels": roofs,
            "fp4_probe": probe,
            "kernels_us": {k: round(v, 2) for k, v in kern.items()},
            "kernels_us_note": "CUDA graph of back-to-back launches cycling over input copies (> 2 x L2 in total), replayed 20 "
                               "times: kernel-to-kernel time; step_eager_us = the same step without a graph",
            "bf16_lora_baseline": {"us_per_step": bf16_us, "speedup": bf16_us / (ms_per_step * 1e3),
                                   "how": "torch.matmul (cuBLAS) bf16, frozen W, same shapes, same GPU, same protocol "
                                          "(CUDA graph, back-to-back replays)"},
            "saved4_activations": {
                "wgrad_bf16_x_us": round(kern["wgrad_dA_dBt_us"], 2), "wgrad_saved4_us": round(kern["wgrad_saved4_us"], 2),
                "step_us": round(kern["step_saved4_us"], 2), "step_bf16_x_us": round(kern["step_bf16x_us"], 2),
                "saved_bytes_per_layer_bf16": 2 * M * K, "saved_bytes_per_layer_4bit": int(0.5625 * M * K),
                "note": "NEXT-2: ft_lora_wgrad_q4 takes dA = dequant(Q(X))^T (G B^T) from the codes and scales the "
                        "forward pass wrote, so the bf16 X need not be kept for backward (3.56x fewer saved bytes); "
                        "step_us = ft_linear_fwd + ft_linear_bwd_q4 as a CUDA graph, 100 replays; the headline step follows "
                        "Eq. 4 literally (O-12)"},
            "single_copy_weights": {
                "step_us": round(kern["step_single_copy_us"], 2), "step_two_copies_us": round(kern["step_bf16x_us"], 2),
                "transpose_us": round(kern["transpose_codes_us"], 2),
                "transpose_GBps": round(N * K / (kern["transpose_codes_us"] * 1e-6) / 1e9, 1),
                "weight_bytes_per_layer_two_copies": int(N * K * (0.5 + 0.5 + 2 / 16)),
                "weight_bytes_per_layer_single_copy": int(N * K * (0.5 + 2 / 16)),
                "scratch_bytes_shared_by_all_layers": N * K // 2,
                "note": "NEXT-5 (PAPER.md:102, :197): one copy of the 4-bit codes per layer; ft_weight_transpose_codes "
                        "rebuilds the codes of Q(R)^T into one scratch buffer before the layer's backward (N K bytes "
                        "of traffic: N K / 2 read + N K / 2 written); both scale layouts (N K / 16 each) stay per "
                        "layer.  The 4-bit MMA takes K-major operands only, so the element transposition cannot be "
                        "left to the tensor core or to TMA"},
            **extra,
            "paper_context": "2.27x step time / 2.25x memory vs BF16 LoRA on RTX 5090 (PAPER.md:7,207); not the target",
            "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cpu_cores(), "kind": "oracle",
                             "sample": "all 4608 tokens of C2, fwd+dgrad+wgrad, mean of 2 passes (%.1f s of CPU work)"
                                       % sum(cpu_times)},
        }
        print(json.dumps(out))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


# ------------------------------------------------------------------ the other BASELINE.json configs
def sweep(B, prepare, dev, graph_us, peaks, full=False):
    """C4 (quantizer-only sweep; always) and, with --sweep, C1 / C3 / C5 layer timings.  Inputs are
    torch-generated on the device with the configs' shapes (N(0,1) with 1 % channels x50; gradients
    1e-3 N(0,1)): throughput does not depend on the values; parity on these shapes is in tests/."""
    import torch
    g = torch.Generator(device=dev)
    g.manual_seed(3)

    def acts(rows, cols, grad=False):
        x = torch.randn(rows, cols, device=dev, generator=g)
        if grad:
            return (x * 1e-3).to(torch.bfloat16)
        idx = torch.randperm(cols, device=dev, generator=g)[: max(1, cols // 100)]
        x[:, idx] *= 50.0
        return x.to(torch.bfloat16)

    out = {}
    c4 = []
    for rows, cols in ((4608, 3072), (4608, 12288), (4608, 15360), (9216, 3072)):
        ncopy = max(2, int(300e6 // (rows * cols * 2)) + 1)          # together > 2 x L2: every launch reads HBM
        xs = [acts(rows, cols) for _ in range(ncopy)]
        q = B.QTensor(rows, cols, device=dev)
        ws = B.new_workspace(rows, cols, 0, 32, dev)
        amax = B.ft_tensor_amax(xs[0])
        d = (torch.randn(cols, 32, device=dev, generator=g) * 0.01).to(torch.bfloat16)
        h = torch.empty(rows, 32, dtype=torch.bfloat16, device=dev)
        t_a = graph_us([lambda x=x: B.ft_tensor_amax(x, amax) for x in xs])
        amax = B.ft_tensor_amax(xs[0])
        t_q = graph_us([lambda x=x: B.ft_quantize_blockwise(x, q, tensor_amax=amax, workspace=ws) for x in xs])
        t_p = graph_us([lambda x=x: B.ft_quantize_blockwise(x, q, tensor_amax=amax, down=d, h_out=h, workspace=ws) for x in xs])
        t_f = graph_us([lambda x=x: B.ft_quantize_blockwise(x, q, down=d, h_out=h, workspace=ws) for x in xs])   # a0 + a1, one call
        by = 2.5625 * rows * cols
        byp = by + 4.0 * 32 * rows            # + H (bf16) and the D slices, once per row tile pass: 4 r_t / cols per element
        c4.append({"shape": [rows, cols], "amax_us": round(t_a, 2), "amax_GBps": round(2.0 * rows * cols / t_a / 1e3),
                   "quant_us": round(t_q, 2), "quant_GBps": round(by / t_q / 1e3),
                   "quant_proj32_us": round(t_p, 2), "quant_proj32_GBps": round(byp / t_p / 1e3),
                   "amax_quant_proj32_one_call_us": round(t_f, 2),
                   "frac_of_hbm": round(by / t_q / 1e3 / peaks["hbm"], 3),
                   "frac_of_hbm_proj32": round(byp / t_p / 1e3 / peaks["hbm"], 3),
                   "frac_of_nominal_8TBps_proj32": round(byp / t_p / 1e3 / 8000.0, 3)})
        del xs, q, ws, d, h
        torch.cuda.empty_cache()
    out["C4_quantizer_sweep"] = {"bytes_per_element": 2.5625, "hbm_peak_GBps": peaks["hbm"],
                                 "note": "amax given (except the one-call column); each call captured back to back in one "
                                         "CUDA graph over input copies that together exceed 2 x L2, replayed 20 times: "
                                         "kernel-to-kernel time of k_quantize_fused (+ k_finalize_h with the projection)",
                                 "cases": c4}
    if not full:
        return out

    def layer_case(M, K, N, r_s, r):
        r_t = r_s + r
        X, G = acts(M, K), acts(M, N, grad=True)
        W = (torch.randn(N, K, device=dev, generator=g) * 0.02).to(torch.bfloat16)
        D_f = (torch.randn(K, r_t, device=dev, generator=g) * 0.01).to(torch.bfloat16)
        U_t = (torch.randn(N, r_t, device=dev, generator=g) * 0.01).to(torch.bfloat16)
        layer = B.Layer(W, D_f, U_t, r_s, r, tokens=M)
        y = torch.empty(M, N, dtype=torch.bfloat16, device=dev)
        dx = torch.empty(M, K, dtype=torch.bfloat16, device=dev)
        h = torch.empty(M, r_t, dtype=torch.bfloat16, device=dev)
        p = torch.empty(M, r_t, dtype=torch.bfloat16, device=dev)
        ws = B.new_workspace(M, max(K, N), max(K, N), r_t, dev)
        qx, qg = B.QTensor(M, K, device=dev), B.QTensor(M, N, device=dev)
        dA = torch.empty(K, r, dtype=torch.float32, device=dev)
        dBt = torch.empty(N, r, dtype=torch.float32, device=dev)

        def step():
            B.ft_linear_fwd(layer, X, y, h, qx, ws)
            B.ft_linear_bwd(layer, X, G, h, dx, p, dA, dBt, qg, ws)
        ours = graph_us([step], 20)
        A_, B_ = D_f[:, r_s:].contiguous(), U_t[:, r_s:].t().contiguous()

        def bf16():
            xa = X @ A_
            X @ W.t() + xa @ B_
            gb = G @ B_.t()
            G @ W + gb @ A_.t()
            X.t() @ gb
            xa.t() @ G
        base = graph_us([bf16], 5)            # the same protocol for the baseline: CUDA graph, back-to-back replays
        return ours, base

    out["fusion_ablation_C2"] = fusion_ablation(B, dev, acts, g)
    out["mlp_fusion_C3"] = mlp_fusion(B, dev, acts, g, graph_us)
    torch.cuda.empty_cache()
    cfgs = {"C1": (256, 3072, 3072, 32, 16), "C3u": (4608, 3072, 12288, 32, 64), "C3d": (4608, 12288, 3072, 32, 64)}
    out["configs"] = {}
    for name, (M, K, N, r_s, r) in cfgs.items():
        ours, base = layer_case(M, K, N, r_s, r)
        out["configs"][name] = {"M": M, "K": K, "N": N, "r_s": r_s, "r": r, "step_us": round(ours, 1),
                                "TFLOPs": round(4.0 * M * N * K / ours / 1e6, 1), "bf16_lora_us": round(base, 1),
                                "speedup_vs_bf16_lora": round(base / ours, 2)}
        torch.cuda.empty_cache()
    from paper_2607_05711_b200 import synth
    tot_ours = tot_base = tot_flop = 0.0
    rows = []
    for name, count, M, K, N in synth.C5_LAYERS:
        ours, base = layer_case(M, K, N, 32, 32)
        tot_ours += count * ours
        tot_base += count * base
        tot_flop += count * 4.0 * M * N * K
        rows.append({"layer": name, "count": count, "M": M, "K": K, "N": N, "step_us": round(ours, 1),
                     "bf16_lora_us": round(base, 1)})
        torch.cuda.empty_cache()
    out["C5_dit_linear_layers"] = {"layers": 228, "distinct_shapes": rows, "how": "each distinct (M,K,N) timed once "
                                   "(CUDA graph, 20 replays back to back; the bf16 baseline the same way) and multiplied by "
                                   "its count",
                                   "fwd_bwd_ms": round(tot_ours / 1e3, 2), "TFLOPs": round(tot_flop / tot_ours / 1e6, 1),
                                   "bf16_lora_ms": round(tot_base / 1e3, 2),
                                   "speedup_vs_bf16_lora": round(tot_base / tot_ours, 2)}
    return out


def mlp_fusion(B, dev, acts, g, graph_us):
    """NEXT-1 ("further fusing the MLP components provides an additional 1.10x"): the FLUX-shaped
    MLP pair of BASELINE.json configs[2] (M=4608, 3072 -> 12288 -> GeLU -> 3072, r_s=32, r=64), forward and backward,
    with and without the MLP fusion.  Unfused = the two LoRA-fused layers with bf16 Y1 and Z in HBM and the GeLU
    (forward and backward) as torch elementwise kernels.  Fused = ft_mlp_fwd (GeLU, FC2's quantize and
    down-projection in FC1's GEMM epilogue; Y1 and Z kept as NVFP4 only) and a backward on the 4-bit saved
    activations: ft_linear_bwd_q4(FC2), ft_gelu_bwd_q4, ft_linear_bwd_q4(FC1)."""
    import torch
    import torch.nn.functional as F
    M, K, N1, N2, r_s, r = 4608, 3072, 12288, 3072, 32, 64
    r_t = r_s + r
    X, G2 = acts(M, K), acts(M, N2, grad=True)

    def mk(n, k, ntile):
        W = (torch.randn(n, k, device=dev, generator=g) * 0.02).to(torch.bfloat16)
        D = (torch.randn(k, r_t, device=dev, generator=g) * 0.01).to(torch.bfloat16)
        U = (torch.randn(n, r_t, device=dev, generator=g) * 0.01).to(torch.bfloat16)
        return B.Layer(W, D, U, r_s, r, ntile=ntile)
    fc1, fc2 = mk(N1, K, 224), mk(N2, N1, 224)
    # the same FC1 with its forward scales cut to 192-wide tiles (what ft_mlp_fwd's GEMM runs); weights are random, so
    # a second random matrix of the same shape serves the timing
    fc1f = mk(N1, K, 192)
    bf = torch.bfloat16
    y1 = torch.empty(M, N1, dtype=bf, device=dev); z = torch.empty_like(y1); dz = torch.empty_like(y1); dy1 = torch.empty_like(y1)
    y2 = torch.empty(M, N2, dtype=bf, device=dev); dx = torch.empty(M, K, dtype=bf, device=dev)
    h1 = torch.empty(M, r_t, dtype=bf, device=dev); h2 = torch.empty_like(h1); p1 = torch.empty_like(h1); p2 = torch.empty_like(h1)
    qx, qz, qy1 = B.QTensor(M, K, device=dev), B.QTensor(M, N1, device=dev), B.QTensor(M, N1, device=dev)
    qg2, qg1 = B.QTensor(M, N2, device=dev), B.QTensor(M, N1, device=dev)
    ws = B.new_mlp_workspace(M, max(K, N1), N1, r_t, r_t, dev)
    ws2 = B.new_workspace(M, N1, N1, r_t, dev)
    dA1 = torch.empty(K, r, dtype=torch.float32, device=dev); dB1 = torch.empty(N1, r, dtype=torch.float32, device=dev)
    dA2 = torch.empty(N1, r, dtype=torch.float32, device=dev); dB2 = torch.empty(N2, r, dtype=torch.float32, device=dev)
    za = torch.empty(1, device=dev); ya = torch.empty(1, device=dev)

    def fwd_unfused():
        B.ft_linear_fwd(fc1, X, y1, h1, qx, ws2)
        torch.ops.aten.gelu.out(y1, approximate="tanh", out=z)
        B.ft_linear_fwd(fc2, z, y2, h2, qz, ws2)

    def bwd_unfused():
        B.ft_linear_bwd(fc2, z, G2, h2, dz, p2, dA2, dB2, qg2, ws2)
        torch.ops.aten.gelu_backward.grad_input(dz, y1, approximate="tanh", grad_input=dy1)
        B.ft_linear_bwd(fc1, X, dy1, h1, dx, p1, dA1, dB1, qg1, ws2)
    fwd_unfused()
    torch.cuda.synchronize()
    za.copy_(z.float().abs().max()); ya.copy_(y1.float().abs().max())     # "the previous step's" amax

    def fwd_fused():
        B.ft_mlp_fwd(fc1f, fc2, X, za, ya, y2, h1, h2, qx, qz, qy1, ws)

    def bwd_fused():
        B.ft_linear_bwd_q4(fc2, qz, G2, h2, dz, p2, dA2, dB2, qg2, ws2)
        B.ft_gelu_bwd_q4(dz, qy1, dz)
        B.ft_linear_bwd_q4(fc1, qx, dz, h1, dx, p1, dA1, dB1, qg1, ws2)
    res = {}
    res["fwd_unfused_us"] = round(graph_us([fwd_unfused], 10), 1)
    res["fwd_fused_us"] = round(graph_us([fwd_fused], 10), 1)
    res["fwd_bwd_unfused_us"] = round(graph_us([lambda: (fwd_unfused(), bwd_unfused())], 10), 1)
    res["fwd_bwd_fused_us"] = round(graph_us([lambda: (fwd_fused(), bwd_fused())], 10), 1)
    res["fwd_speedup"] = round(res["fwd_unfused_us"] / res["fwd_fused_us"], 3)
    res["fwd_bwd_speedup"] = round(res["fwd_bwd_unfused_us"] / res["fwd_bwd_fused_us"], 3)
    res["activation_bytes_kept_unfused"] = 2 * M * K + 2 * 2 * M * N1       # bf16 X, Y1, Z
    res["activation_bytes_kept_fused"] = int(0.5625 * (M * K + 2 * M * N1))  # Q(X), Q(Y1), Q(Z)
    res["note"] = ("CUDA graphs, 10 replays; unfused = two LoRA-fused layers + torch GeLU kernels, bf16 Y1 and Z in HBM; fused = "
                   "ft_mlp_fwd + backward on the 4-bit saved activations (delayed-scaling amax for Q(Z), Q(Y1): reading "
                   "O-16); paper (other GPUs, whole DiT): MLP fusion +1.10x (PAPER.md:245)")
    return res


def fusion_ablation(B, dev, acts, g):
    """The shape of the paper's kernel-fusion experiment (Fig. 9) on this GPU, C2 shapes:
    the same 4-bit GEMM kernels with NOTHING fused around them -- separate amax and quantize launches, the
    down- and up-projections as cuBLAS bf16 GEMMs, the branch sum as an elementwise add, the two LoRA
    gradients as one launch -- against the fused path bench.py times.  Timing only (the unfused arm does
    not pre-scale H, so its numbers are not the library's)."""
    import torch
    M, K, N, r_s, r = 4608, 3072, 9216, 32, 32
    r_t = r_s + r
    X, G = acts(M, K), acts(M, N, grad=True)
    W = (torch.randn(N, K, device=dev, generator=g) * 0.02).to(torch.bfloat16)
    D_f = (torch.randn(K, r_t, device=dev, generator=g) * 0.01).to(torch.bfloat16)
    U_t = (torch.randn(N, r_t, device=dev, generator=g) * 0.01).to(torch.bfloat16)
    layer = B.Layer(W, D_f, U_t, r_s, r, tokens=M)
    y = torch.empty(M, N, dtype=torch.bfloat16, device=dev)
    dx = torch.empty(M, K, dtype=torch.bfloat16, device=dev)
    h = torch.empty(M, r_t, dtype=torch.bfloat16, device=dev)
    p = torch.empty(M, r_t, dtype=torch.bfloat16, device=dev)
    ws = B.new_workspace(M, max(K, N), max(K, N), r_t, dev)
    qx, qg = B.QTensor(M, K, device=dev), B.QTensor(M, N, device=dev)
    dA = torch.empty(K, r, dtype=torch.float32, device=dev)
    dBt = torch.empty(N, r, dtype=torch.float32, device=dev)
    ax, ag = torch.empty(1, device=dev), torch.empty(1, device=dev)
    U_f, D_t = U_t.t().contiguous(), D_f.t().contiguous()

    def unfused():
        B.ft_tensor_amax(X, ax)
        B.ft_quantize_blockwise(X, qx, tensor_amax=ax, workspace=ws)
        hh = X @ D_f
        B.ft_gemm4(qx, layer.r_kmajor, None, None, y)
        y.add_(hh @ U_f)
        B.ft_tensor_amax(G, ag)
        B.ft_quantize_blockwise(G, qg, tensor_amax=ag, workspace=ws)
        pp = G @ U_t
        B.ft_gemm4(qg, layer.r_nmajor, None, None, dx)
        dx.add_(pp @ D_t)
        B.ft_lora_wgrad(layer, X, G, hh, pp, dA, dBt)

    def fused():
        B.ft_linear_fwd(layer, X, y, h, qx, ws)
        B.ft_linear_bwd(layer, X, G, h, dx, p, dA, dBt, qg, ws)

    res = {}
    for name, fn in (("unfused_4bit_us", unfused), ("fused_us", fused)):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        gr = torch.cuda.CUDAGraph()
        with torch.cuda.graph(gr):
            fn()
        for _ in range(3):
            gr.replay()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(20):
            gr.replay()
        b.record()
        torch.cuda.synchronize()
        res[name] = round(a.elapsed_time(b) / 20 * 1e3, 1)
    res["fusion_speedup"] = round(res["unfused_4bit_us"] / res["fused_us"], 2)
    res["note"] = ("both arms as CUDA graphs; unfused = k_amax, quantize without projection, cuBLAS bf16 down-/up-"
                   "projections, elementwise adds, the same 4-bit GEMM kernel: a TIMING shape only, its outputs are "
                   "UNCHECKED (it does not pre-scale H, so its numbers are not the library's); paper (other GPUs, whole "
                   "DiT): LoRA fusion 1.82x (PAPER.md:245)")
    return res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--eager", action="store_true", help="no CUDA graph for the timed steps")
    ap.add_argument("--sweep", action="store_true", help="(default) also time C4, C1, C3, the fusion ablation and the "
                                                         "C5 layer list: adds ~25 s")
    ap.add_argument("--c4-only", dest="c4_only", action="store_true", help="of the other configs, time only the C4 sweep")
    ap.add_argument("--no-sweep", dest="no_sweep", action="store_true", help="time the C2 step only")
    ap.add_argument("--probe-seconds", dest="probe_seconds", type=float, default=1.5,
                    help="duration of the sustained FP4 tensor-core probe (0 = skip)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
