#!/usr/bin/env python
"""bench.py — the steady-state pipelined step of BASELINE.json configs[2] on N B200s (replicas).

A "step" is one pass of the whole hot path over one packed batch: the 276-row
prefill of a new frame + 6 single-row decodes of the in-flight frames through the 32-layer Llama-2-7B-shaped stack,
then the LM head on the 7 prediction rows.  In steady state one step completes one action frame (7 action tokens).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Prints ONE JSON line (see DESIGN.md "Measurement" for every field).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

L_P, K_STAGES, R_REGIONS, CAPACITY = 276, 7, 8, 512      # 256 patch + 20 prompt tokens, K = 7 action tokens
SEED = 2
# DRAM bytes per gemm_tcgen05_kernel launch (dram__bytes_read.sum + dram__bytes_write.sum, averaged over the launches of
# a steady step; cold caches): profiles/launches_r1.md.  Algorithmic weight bytes per launch: 102.8 MB.
GEMM_TRAFFIC_BYTES_PER_LAUNCH = 107.2e6
WORKLOAD = "cfg3: 32-layer Llama-2-7B shape, steady pipelined step = 276-row prefill + 6 decodes (ctx 277..282) + LM head on 7 rows"


# ---------------------------------------------------------------------------------------------- work model
def step_work(cfg, segs, n_logit_rows):
    """Algorithmic FLOPs and bytes of one step (SURVEY.md 8(d) / DESIGN.md "Roofline")."""
    D, F, V, Lyr, H, hd = cfg.d_model, cfg.ffn, cfg.vocab, cfg.n_layers, cfg.n_heads, cfg.head_dim
    T = sum(s[3] for s in segs)
    p_layer = 4 * D * D + 3 * D * F
    sum_ctx_rows = sum(sum(range(s[2] + 1, s[2] + s[3] + 1)) for s in segs)       # sum over rows of (pos+1)
    sum_ctx_segs = sum(s[2] + s[3] for s in segs)
    gemm_flops = 2 * T * Lyr * p_layer + 2 * n_logit_rows * V * D
    attn_flops = 4 * D * Lyr * sum_ctx_rows
    kv_row = 2 * H * hd * 2
    w_bytes = 2 * (Lyr * p_layer + (2 * Lyr + 1) * D) + (2 * V * D if n_logit_rows else 0)
    kv_read = kv_row * Lyr * sum_ctx_segs
    kv_write = kv_row * Lyr * T
    io = 2 * T * D + 4 * T * D + 4 * n_logit_rows * V
    return {"T": T, "gemm_flops": gemm_flops, "attn_flops": attn_flops, "flops": gemm_flops + attn_flops,
            "weight_bytes": w_bytes, "kv_read_bytes": kv_read, "kv_write_bytes": kv_write,
            "bytes": w_bytes + kv_read + kv_write + io}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "tf_burst": d["bf16_tflops"], "tf_sustained": d["bf16_tflops_sustained"],
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "tf_burst": 1590.0, "tf_sustained": 1400.0, "source": "fallback"}


# ---------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
        sm = sorted(int(float(r[0])) for r in self.rows if r and r[0].replace(".", "").isdigit())
        mx = [int(float(r[1])) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 7 for i in range(4) if r[3 + i].lower() == "active"})
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# ---------------------------------------------------------------------------------------------- reference arm
def bench_config(layers=32):
    """The `config` object of the bench line; the reference arm prints the same one (same workload, same keys)."""
    return {"workload": WORKLOAD if layers == 32 else f"DEBUG {layers}-layer slice of " + WORKLOAD,
            "precision": "bf16-valued weights stored as fp16 (af_convert_bf16_to_fp16 at load; exact for 2^-14 <= |w| <= "
                         "65504, smaller values round to fp16 subnormals, abs err <= 2^-25), fp16 activations and KV "
                         "ring, fp32 accumulate / residual / logits (tcgen05 kind::f16)",
            "packed_rows": L_P + K_STAGES - 1, "ring": f"{R_REGIONS} regions x {CAPACITY}",
            "multi_gpu": "independent replicas",
            "l2": "inputs larger than L2 (13.2 GB of weights streamed per step vs 126 MB L2)"}


def oracle_frame(orc, cfg, seed, frame, torch, I):
    """One WHOLE frame of the paper's Baseline schedule through the oracle as it stands: the 276-row prefill,
    then the 6 decodes one by one (each alone, unpacked), then the LM head on the 7 prediction rows.  Returns seconds."""
    n_dec = K_STAGES - 1
    e = I.make_embeds(cfg, seed, frame, L_P + n_dec)
    t0 = time.perf_counter()
    orc.reset(0)
    hid = [orc.step([(0, 0, 0, L_P)], e[:L_P])[-1:]]
    for s in range(n_dec):
        hid.append(orc.step([(0, 1, L_P + s, 1)], e[L_P + s:L_P + s + 1]))
    orc.logits(torch.cat(hid), list(range(1 + n_dec)))
    return time.perf_counter() - t0


def oracle_cores():
    return max(1, (os.cpu_count() or 4) - 2)       # leave two cores free: an oversubscribed OpenMP pool collapses


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only).  A step is one whole 32-layer frame
    (nothing is extrapolated); only when steps + warmup whole frames would not end within ~4 minutes is the layer count
    of every step's sample reduced, and the line then says so."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import torch
    from oracle import af_oracle as O
    from paper_2512_20276_b200 import inputs as I
    cores = oracle_cores()
    torch.set_num_threads(cores)
    warmup = max(1, args.warmup)
    cfg = I.cfg_7b_layers(args.layers)
    hw = I.make_weights(cfg, SEED, threads=max(4, os.cpu_count() or 8))
    orc = O.Oracle(cfg, hw, torch.float32)
    t_first = oracle_frame(orc, cfg, SEED, 0, torch, I)              # warm-up frame 1 (also sizes the run)
    n_layers = cfg.n_layers
    budget = 240.0
    if t_first * (args.steps + warmup) > budget and n_layers > 1:
        n_layers = max(1, int(cfg.n_layers * budget / (t_first * (args.steps + warmup))))
        cfg_s = I.cfg_7b_layers(n_layers)
        orc = O.Oracle(cfg_s, {"layers": hw["layers"][:n_layers], "g_final": hw["g_final"], "w_lm": hw["w_lm"]}, torch.float32)
    else:
        cfg_s = cfg
    for i in range(1, warmup):
        oracle_frame(orc, cfg_s, SEED, i, torch, I)
    t0 = time.perf_counter()
    for i in range(args.steps):
        oracle_frame(orc, cfg_s, SEED, warmup + i, torch, I)
    step_s = (time.perf_counter() - t0) / args.steps
    fps = 1.0 / step_s
    sample = (f"{n_layers} of {cfg.n_layers} layers; every step is one whole frame through the oracle (276-row prefill + 6 "
              f"sequential single-row decodes + LM head on 7 rows), {args.steps} timed frames after {warmup} warm-up frames")
    if n_layers != cfg.n_layers:
        sample += f"; REDUCED SAMPLE: value and ms_per_step are those of the {n_layers}-layer frame actually run, not of the full stack"
    line = {"impl": "reference", "metric": "action_frames_per_s", "value": fps, "unit": "frames/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_s * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": bench_config(args.layers),
            "reference": "unpacked sequential fp32 CPU oracle (oracle/af_oracle.py, Python + torch CPU ops), as it stands",
            "packed_tok_per_s": fps * (L_P + K_STAGES - 1),
            "cpu_baseline": {"value": fps, "unit": "frames/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": fps, "unit": "frames/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------- library GEMM context
def run_library_gemm(args, emit=True):
    """Context for roofline.frac, not a product path: what the vendor library (cuBLAS through torch.matmul, fp16 in,
    fp32 accumulate) reaches on the step's own projection shapes, T = 282 packed rows against [out, in] weights, with a
    different weight matrix every call (8 per shape, > L2 in total) as in a real step.  Same GPU, same process, CUDA
    events around 64 back-to-back calls after 16 warm-up calls.  Prints one JSON line; summarised in profiles/."""
    import torch
    if emit:
        torch.cuda.set_device(0)
    T, D, F = L_P + K_STAGES - 1, 4096, 11008
    shapes = [("qkv", 3 * D, D), ("o", D, D), ("gate_up", 2 * F, D), ("down", D, F)]
    g = torch.Generator(device="cuda").manual_seed(SEED)
    ws = {n: [(0.02 * torch.randn(o, k, generator=g, device="cuda")).half() for _ in range(8)] for n, o, k in shapes}
    xs = {n: torch.randn(T, k, generator=g, device="cuda").half() for n, o, k in shapes}

    def layers(n_layers, events=None):
        for l in range(n_layers):
            for name, _, _ in shapes:
                if events is not None:
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                torch.matmul(xs[name], ws[name][l % 8].t())
                if events is not None:
                    e1.record()
                    events[name].append((e0, e1))

    sampler = ClockSampler(torch.cuda.current_device())
    layers(32 * 300)                                     # ~1.3 s: reach the power-capped clock a long step runs at
    torch.cuda.synchronize()
    sampler.start()
    # (a) back to back, as a library user would chain them: one pair of events around 32 x 64 layers
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    layers(32 * 64)
    e1.record()
    torch.cuda.synchronize()
    chained_us = e0.elapsed_time(e1) / (32 * 64) * 1e3
    # (b) per launch events, the way bench.py's kernel_ms_per_step times this library's own GEMM launches
    ev = {n: [] for n, _, _ in shapes}
    layers(32 * 20, ev)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    out = {}
    for name, n_out, k in shapes:
        us = sum(a.elapsed_time(b) for a, b in ev[name]) / len(ev[name]) * 1e3
        out[name] = {"us_per_call": us, "tflops": 2.0 * T * n_out * k / us / 1e6, "weight_gbs": 2.0 * n_out * k / us / 1e3}
    layer_us = sum(v["us_per_call"] for v in out.values())
    flops = 2.0 * T * (4 * D * D + 3 * D * F)
    res = {"what": "cuBLAS (torch.matmul fp16) on the step's projection shapes, T = 282, cold weights",
           "per_shape_event_timed": out, "layer_gemm_us_event_timed": layer_us,
           "layer_tflops_event_timed": flops / layer_us / 1e6, "layer_gemm_us_chained": chained_us,
           "layer_tflops_chained": flops / chained_us / 1e6, "clocks": clocks}
    if emit:
        print(json.dumps(res), flush=True)
    return res


# ---------------------------------------------------------------------------------------------- GEMM timeline
def run_gemm_timeline(args):
    """Report for profiles/: af_debug_trace's %globaltimer stamps of the GEMM launches of two steady cfg3 steps on a
    2-layer slice (same shapes and launch configuration as the bench step), as min / median / max over CTAs in us
    after the launch's first CTA starts.  One markdown table row per launch."""
    import ctypes as C
    import numpy as np
    import torch
    from paper_2512_20276_b200 import binding, inputs as I
    torch.cuda.set_device(0)
    L = binding.load_library()
    cfg = I.cfg_7b_layers(2)
    W = binding.Weights(cfg, I.make_weights(cfg, SEED, threads=16))
    ring = binding.Ring(cfg, R_REGIONS, CAPACITY, max_rows=288)

    def step(t):
        ring.reset_slot(t % R_REGIONS, -1)
        segs = I.steady_schedule(t, L_P, K_STAGES, R_REGIONS)
        ring.packed_forward(W, I.make_embeds(cfg, SEED, t, I.total_rows(segs)).cuda(), segs)

    for t in range(12):
        step(t)
    torch.cuda.synchronize()
    L.af_debug_trace.argtypes, L.af_debug_trace.restype = [C.c_int], C.c_int
    L.af_debug_trace_read.argtypes, L.af_debug_trace_read.restype = [C.c_void_p, C.c_void_p], C.c_int
    L.af_debug_trace(1)
    step(12)
    step(13)
    torch.cuda.synchronize()
    st, meta = np.zeros((16, 160, 32), dtype=np.int64), np.zeros((16, 2), dtype=np.int32)
    L.af_debug_trace_read(st.ctypes.data, meta.ctypes.data)
    L.af_debug_trace(0)
    cols = [("released (producer past griddepcontrol.wait)", 25), ("producer requested its last stage", 26),
            ("piece 0: accumulator ready", 3), ("piece 0: drained", 5), ("piece 1: accumulator ready", 7),
            ("piece 1: fix-up loaded", 8), ("piece 1: drained", 9)]
    names = ["QKV", "O", "gate/up", "down", "LM head"]
    print("| launch | grid | first CTA .. last CTA start | " + " | ".join(c[0] for c in cols) + " |")
    print("|---|---|---|" + "---|" * len(cols))
    for li in range(16):
        cat, grid = int(meta[li][0]), int(meta[li][1])
        if grid <= 0 or li >= 8:
            continue
        s = st[li, :grid]
        t0 = s[:, 0][s[:, 0] > 0].min()

        def rel(col):
            v = s[:, col].astype(np.float64)
            v[s[:, col] == 0] = np.nan
            v = (v - t0) / 1e3
            return "-" if np.all(np.isnan(v)) else f"{np.nanmin(v):.1f} / {np.nanmedian(v):.1f} / {np.nanmax(v):.1f}"
        print(f"| {names[cat] if cat < 5 else cat} | {grid} | {rel(0)} | " + " | ".join(rel(c[1]) for c in cols) + " |")


# ---------------------------------------------------------------------------------------------- cfg5 sweep
def run_sweep(args):
    """BASELINE.json configs[4]: concurrent decodes x prefill length at the 7B shape.  Prints one markdown table row per
    grid point (step latency, packed tok/s, achieved HBM GB/s = algorithmic bytes / latency, tensor TFLOP/s, fraction
    of the point's roofline at the measured peaks).  Not the bench line; a report for profiles/."""
    import torch
    from paper_2512_20276_b200 import binding, inputs as I
    torch.cuda.set_device(0)
    cfg = I.cfg_7b_layers(args.layers)
    hw = I.make_weights(cfg, 4, threads=max(4, os.cpu_count() or 8))
    W = binding.Weights(cfg, hw)
    # --chunks: SURVEY.md 8(f) row f2, the paper's longer action chunks (section 4.3, Fig. 5): K - 1 decode segments
    # ride on one 276-row prefill, K in {7, 16, 24, 32}; decode j's history is the first 276 + j rows of H as in cfg5
    max_dec = 31 if args.chunks else 15
    Rr, Cc = max_dec + 2, 1024 if not args.chunks else 512
    ring = binding.Ring(cfg, Rr, Cc, max_rows=544)
    H = I.make_embeds(cfg, 4, 1, 276 + max_dec).cuda()
    E = I.make_embeds(cfg, 4, 0, 512).cuda()
    for j in range(max_dec):
        ring.packed_forward(W, H[:276 + j].contiguous(), [(j + 1, 0, 0, 276 + j)])
    peaks = load_peaks()
    hidden = torch.empty(544, cfg.d_model, dtype=torch.float32, device="cuda")
    print("| decodes | prefill | T | ms/step | packed tok/s | HBM GB/s (algorithmic) | TFLOP/s | roofline ms (measured peaks) | frac |")
    print("|---|---|---|---|---|---|---|---|---|")
    grid = [(n, 276) for n in (6, 15, 23, 31)] if args.chunks else \
           [(n, p) for n in (0, 1, 3, 6, 10, 15) for p in (0, 128, 276, 512)]
    for n_dec, p_len in grid:
        if True:
            if n_dec == 0 and p_len == 0:
                continue
            segs, rows = [], []
            if p_len:
                segs.append((0, 0, 0, p_len)); rows.append(E[:p_len])
            for j in range(n_dec):
                segs.append((j + 1, 1, 276 + j, 1)); rows.append(H[276 + j:277 + j])
            x = torch.cat(rows).contiguous()

            def one():
                ring.reset_slot(0, 0)
                for j in range(max_dec):
                    ring.set_len(j + 1, 276 + j)
                ring.packed_forward(W, x, segs, hidden_out=hidden[:x.shape[0]])
            for _ in range(3):
                one()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(args.steps):
                one()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / args.steps
            wk = step_work(cfg, segs, 0)
            roof = max(wk["bytes"] / (peaks["hbm_gbs"] * 1e9), wk["flops"] / (peaks["tf_sustained"] * 1e12)) * 1e3
            print(f"| {n_dec} | {p_len} | {wk['T']} | {ms:.3f} | {wk['T'] / ms * 1e3:.0f} | {wk['bytes'] / ms / 1e6:.0f} | "
                  f"{wk['flops'] / ms / 1e9:.0f} | {roof:.3f} | {roof / ms:.2f} |", flush=True)


# ---------------------------------------------------------------------------------------------- our arm
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layers", type=int, default=32, help="debug only: fewer layers (the line then says so)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="print the cfg5 scheduling-shape sweep table instead of the bench line")
    ap.add_argument("--chunks", action="store_true", help="with --sweep: the longer-action-chunk points K = 7, 16, 24, 32 (276-row prefill + K - 1 decodes)")
    ap.add_argument("--library-context", action="store_true", help="add roofline.library_same_shapes: cuBLAS on the step's four projection shapes, same run (context, ~1.5 s of library GEMMs; off by default so that the bench line runs only the product)")
    ap.add_argument("--gemm-timeline", action="store_true", help="report only: af_debug_trace timeline of the GEMM launches of a steady step (markdown table)")
    ap.add_argument("--library-gemm", action="store_true", help="context only: cuBLAS on the step's projection shapes (one JSON line)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.library_gemm:
        return run_library_gemm(args)
    if args.gemm_timeline:
        return run_gemm_timeline(args)
    if args.sweep or args.chunks:
        return run_sweep(args)

    import torch
    import torch.distributed as dist
    from paper_2512_20276_b200 import binding, inputs as I, replicas

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    warmup = max(3, args.warmup)
    cfg = I.cfg_7b_layers(args.layers)
    hw = I.make_weights(cfg, SEED, threads=max(4, os.cpu_count() or 8))
    W = binding.Weights(cfg, hw)
    T = L_P + K_STAGES - 1
    ring = binding.Ring(cfg, R_REGIONS, CAPACITY, max_rows=288)
    n_buf = 8
    e_host = [I.make_embeds(cfg, SEED, t, T).pin_memory() for t in range(n_buf)]
    e_dev = [e.cuda() for e in e_host]
    hidden = torch.empty(T, cfg.d_model, dtype=torch.float32, device="cuda")
    logits = torch.empty(K_STAGES, cfg.vocab, dtype=torch.float32, device="cuda")
    logits_host = torch.empty(K_STAGES, cfg.vocab, dtype=torch.float32).pin_memory()
    e_stage = torch.empty(T, cfg.d_model, dtype=torch.bfloat16, device="cuda")
    stream = torch.cuda.current_stream()
    tau = [0]

    def step(e):
        t = tau[0]
        ring.reset_slot(t % R_REGIONS, -1)                       # recycle the evicted request's region
        segs = I.steady_schedule(t, L_P, K_STAGES, R_REGIONS)
        n = I.total_rows(segs)
        ring.packed_forward(W, e[:n], segs, hidden_out=hidden)
        rows = I.prediction_rows(segs)
        ring.logits_rows(W, hidden, rows, logits_out=logits)
        tau[0] = t + 1

    def barrier():
        replicas.barrier()
        torch.cuda.synchronize()

    for _ in range(K_STAGES - 1 + warmup):                       # pipeline fill + warm-up (untimed)
        step(e_dev[tau[0] % n_buf])
    segs_steady = I.steady_schedule(tau[0], L_P, K_STAGES, R_REGIONS)
    work = step_work(cfg, segs_steady, K_STAGES)

    sampler = ClockSampler(local)
    sampler.start()
    # ---- timed region 1: inputs resident in HBM ----
    launches0 = binding.launch_count()
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        step(e_dev[tau[0] % n_buf])
    ev1.record(stream)
    barrier()
    ms_dev = ev0.elapsed_time(ev1)
    launches = binding.launch_count() - launches0
    # ---- timed region 2: end to end through the public API with host buffers ----
    barrier()
    ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev2.record(stream)
    for _ in range(args.steps):
        e_stage.copy_(e_host[tau[0] % n_buf], non_blocking=True)  # H2D of this step's packed embeddings
        step(e_stage)
        logits_host.copy_(logits, non_blocking=True)             # D2H of this step's logits rows
    ev3.record(stream)
    barrier()
    ms_e2e = ev2.elapsed_time(ev3)
    # ---- timed region 3: the same loop closed on the device - the decode rows of step t + 1 are
    #      af_embed_rows(af_argmax_rows(logits of step t)); only the prefill rows come from the host and only the 7
    #      tokens go back.  The embedding table is synthetic (seeded), like every other input. ----
    table = (0.5 * torch.randn(cfg.vocab, cfg.d_model, generator=torch.Generator().manual_seed(SEED + 7))).to(torch.bfloat16).cuda()
    tokens = torch.zeros(K_STAGES, dtype=torch.int32, device="cuda")
    tokens_host = torch.empty(K_STAGES, dtype=torch.int32).pin_memory()
    for timed in (False, True):
        barrier()
        ev4, ev5 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev4.record(stream)
        for _ in range(args.steps if timed else 3):
            e_stage[:L_P].copy_(e_host[tau[0] % n_buf][:L_P], non_blocking=True)   # H2D: the new frame's prefill rows
            binding.embed_rows(table, tokens[:K_STAGES - 1], out=e_stage[L_P:T])   # decode rows: last tokens, on device
            step(e_stage)
            tokens.copy_(binding.argmax_rows(logits))
            tokens_host.copy_(tokens, non_blocking=True)                           # D2H: 7 action tokens
        ev5.record(stream)
        barrier()
    ms_loop = ev4.elapsed_time(ev5)
    # ---- timed region 4 (f1, second half): af_loop_* - segment table, ring bookkeeping and A_sequences advanced on the
    #      device, the steady step replayed as ONE CUDA graph; the host copies the new frame's prefill rows in and the
    #      completed frame's 7 tokens out, and never synchronises inside the region ----
    ring2 = binding.Ring(cfg, R_REGIONS, CAPACITY, max_rows=288)
    loop = binding.Loop(W, ring2, table, L_P, K_STAGES)
    gs = torch.cuda.Stream()
    frame_host = torch.empty(1 + K_STAGES, dtype=torch.int32).pin_memory()
    with torch.cuda.stream(gs):
        for timed in (False, True):
            barrier()
            ev6, ev7 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            launches_g0 = binding.launch_count()
            ev6.record(gs)
            for i in range(args.steps if timed else K_STAGES - 1 + max(3, warmup)):
                loop.prefill_embeds.copy_(e_host[i % n_buf][:L_P], non_blocking=True)
                loop.step(use_graph=True, stream=gs)
                frame_host.copy_(loop.frame, non_blocking=True)
            ev7.record(gs)
            barrier()
    ms_graph = ev6.elapsed_time(ev7)
    launches_graph = binding.launch_count() - launches_g0
    # ---- per-kernel-class events (separate pass; same steps) ----
    n_prof = min(20, args.steps)
    binding.profile(True)
    for _ in range(n_prof):
        step(e_dev[tau[0] % n_buf])
    prof = binding.profile_read()
    binding.profile(False)
    clocks = sampler.stop()

    ms_dev, ms_e2e, ms_loop, ms_graph = replicas.max_over_ranks([ms_dev, ms_e2e, ms_loop, ms_graph], device="cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = load_peaks()
    ms_step = ms_dev / args.steps
    fps = replicas.whole_job_throughput(args.steps, ms_dev)
    fps_e2e = replicas.whole_job_throughput(args.steps, ms_e2e)
    # the projections run inside layer_chain_kernel ("chain": 4 GEMM phases + the row stages and grid barriers between
    # them per launch) and, for the LM head, gemm_tcgen05_kernel; the per-stage classes stay 0 unless the fallback path ran
    gemm_classes = ["chain", "gemm_qkv", "gemm_o", "gemm_gateup", "gemm_down", "gemm_lm"]
    gemm_ms = sum(prof[k][0] for k in gemm_classes) / n_prof
    gemm_n = sum(prof[k][1] for k in gemm_classes) / n_prof
    all_ms = sum(v[0] for v in prof.values()) / n_prof
    achieved_tf = work["gemm_flops"] / (gemm_ms / 1e3) / 1e12
    roof_hbm_ms = work["bytes"] / (peaks["hbm_gbs"] * 1e9) * 1e3
    roof_tc_ms = work["flops"] / (peaks["tf_sustained"] * 1e12) * 1e3
    roof_nom_ms = max(work["bytes"] / 8e12, work["flops"] / 2.25e15) * 1e3
    line = {
        "metric": "action_frames_per_s", "value": fps, "unit": "frames/s", "n_gpus": world, "steps": args.steps,
        "warmup": warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f16", "data": "synthetic",
        "config": bench_config(args.layers),
        "packed_tok_per_s": fps * T,
        "step_roofline": {"ms_measured_peaks": max(roof_hbm_ms, roof_tc_ms), "hbm_ms": roof_hbm_ms, "tensor_ms": roof_tc_ms,
                          "frac_of_measured": max(roof_hbm_ms, roof_tc_ms) / ms_step,
                          "ms_nominal_8TBs_2.25PF": roof_nom_ms, "frac_of_nominal": roof_nom_ms / ms_step,
                          "peaks": peaks, "flops": work["flops"], "bytes": work["bytes"]},
        "roofline": {"kernel": "layer_chain_kernel (all packed projections of a layer, their row stages and grid barriers) + gemm_tcgen05_kernel (LM head)", "bound": "tensor",
                     "achieved": achieved_tf, "peak": peaks["tf_sustained"], "unit": "TFLOP/s",
                     "frac": achieved_tf / peaks["tf_sustained"],
                     "traffic": GEMM_TRAFFIC_BYTES_PER_LAUNCH if args.layers == 32 else None,
                     "peak_source": peaks["source"] + " sustained bf16 (kernel timed inside a long step)",
                     "launches_per_step": gemm_n, "avg_launch_ms": gemm_ms / max(1, gemm_n),
                     "share_of_step": gemm_ms / all_ms,
                     "weight_stream_gbs": work["weight_bytes"] / (gemm_ms / 1e3) / 1e9},
        "kernel_ms_per_step": {k: v[0] / n_prof for k, v in prof.items()},
        "e2e": {"value": fps_e2e, "unit": "frames/s", "h2d_bytes_per_step": T * cfg.d_model * 2,
                "d2h_bytes_per_step": K_STAGES * cfg.vocab * 4},
        "e2e_device_loop": {"value": replicas.whole_job_throughput(args.steps, ms_loop), "unit": "frames/s",
                            "what": "f1: decode rows = af_embed_rows(af_argmax_rows(previous logits)) on the device",
                            "h2d_bytes_per_step": L_P * cfg.d_model * 2, "d2h_bytes_per_step": K_STAGES * 4},
        "e2e_graph_loop": {"value": replicas.whole_job_throughput(args.steps, ms_graph), "unit": "frames/s",
                           "what": "f1: af_loop_step - device-side segment table / ring bookkeeping / A_sequences, the steady "
                                   "step replayed as one CUDA graph; prefill rows in, the completed frame's tokens out",
                           "h2d_bytes_per_step": L_P * cfg.d_model * 2, "d2h_bytes_per_step": (1 + K_STAGES) * 4,
                           "kernel_nodes_per_step": launches_graph / args.steps},
        "gpu_launches": launches, "clocks": clocks,
    }
    if world == 1 and args.layers == 32 and args.library_context:
        # context, not a product path: the vendor library's GEMMs on the same four shapes, timed the same way
        # (per-launch CUDA events, power-capped clock); see profiles/library_gemm_r1.md
        lib = run_library_gemm(args, emit=False)
        ours_layer_us = sum(prof[k][0] for k in gemm_classes[:5]) / n_prof / cfg.n_layers * 1e3
        line["roofline"]["library_same_shapes"] = {
            "what": "cuBLAS fp16 (torch.matmul) on QKV / O / gate|up / down at T = 282, cold weights, event-timed per launch",
            "layer_gemm_us": lib["layer_gemm_us_event_timed"], "tflops": lib["layer_tflops_event_timed"],
            "frac_of_peak": lib["layer_tflops_event_timed"] / peaks["tf_sustained"],
            "this_library_layer_gemm_us": ours_layer_us, "sm_mhz": lib["clocks"]["sm_mhz"]}
    if not args.no_cpu_baseline:
        # the oracle as it stands, whole 32-layer frames on this box's host cores: 1 warm-up + 2 timed (~5 s each)
        from oracle import af_oracle as O
        torch.set_num_threads(oracle_cores())
        orc = O.Oracle(cfg, hw, torch.float32)
        oracle_frame(orc, cfg, SEED, 0, torch, I)
        n_fr = 2
        frame_s = sum(oracle_frame(orc, cfg, SEED, 1 + i, torch, I) for i in range(n_fr)) / n_fr
        line["cpu_baseline"] = {"value": 1.0 / frame_s, "unit": "frames/s", "cores": torch.get_num_threads(),
                                "kind": "oracle",
                                "sample": f"{cfg.n_layers} of {cfg.n_layers} layers: {n_fr} whole frames timed after 1 warm-up "
                                          "frame (276-row prefill, 6 sequential single-row decodes, LM head on 7 rows), "
                                          "nothing scaled"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
