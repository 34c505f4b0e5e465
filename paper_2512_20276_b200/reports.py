"""Reports for profiles/ (not the bench line): run on one B200, each prints markdown or one JSON line.

    python -m paper_2512_20276_b200.reports --sweep [--steps N]        BASELINE.json configs[4] scheduling-shape sweep
    python -m paper_2512_20276_b200.reports --sweep --chunks           longer action chunks K = 7, 16, 24, 32 (f2)
    python -m paper_2512_20276_b200.reports --sweep --fp8              the same points with AF_WEIGHTS_FP8
    python -m paper_2512_20276_b200.reports --chain-timeline           per-phase timeline of layer_chain_kernel launches
    python -m paper_2512_20276_b200.reports --library-gemm             cuBLAS on the step's projection shapes (context)
    python -m paper_2512_20276_b200.reports --attention-units          the tcgen05 attention units: timeline and step A/B
"""
from __future__ import annotations

import argparse
import json
import os

from .measure import ClockSampler, L_P, K_STAGES, R_REGIONS, CAPACITY, SEED, load_peaks, quantize_on_device, step_work


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


# ---------------------------------------------------------------------------------------------- chain timeline
def run_chain_timeline(args):
    """af_debug_trace's %globaltimer stamps of the layer_chain_kernel launches of one steady cfg3 step on a 3-layer slice
    (same shapes and launch configuration as the bench step): per phase, when its work ended (min / median / max over the
    148 CTAs, us after the launch's first CTA passed griddepcontrol.wait) and when the grid barrier behind it released
    the CTAs; plus the gap between consecutive launches (attention kernel + two kernel boundaries)."""
    import ctypes as C
    import numpy as np
    import torch
    from . import binding, inputs as I
    torch.cuda.set_device(0)
    L = binding.load_library()
    cfg = I.cfg_7b_layers(3)
    hw = I.make_weights(cfg, SEED, threads=16)
    W = binding.WeightsFP8(cfg, quantize_on_device(cfg, hw, torch, I)) if args.fp8 else binding.Weights(cfg, hw)
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
    torch.cuda.synchronize()
    slots = 18
    st, meta = np.zeros((16, 160, slots), dtype=np.int64), np.zeros((16, 2), dtype=np.int32)
    n = L.af_debug_trace_read(st.ctypes.data, meta.ctypes.data)
    L.af_debug_trace(0)
    names = {3: ["x = embeds; RMSNorm", "QKV (layer 0)", "slab reduce + RoPE + ring append"],
             7: ["O proj", "x += slabs; RMSNorm", "gate|up + SiLU*mul", "down proj", "x += slabs; RMSNorm", "QKV (next layer)",
                 "slab reduce + RoPE + ring append"],
             5: ["O proj", "x += slabs; RMSNorm", "gate|up + SiLU*mul", "down proj", "x += slabs (final)"]}
    ends, starts = [], []
    for li in range(min(n, 16)):
        nph, grid = int(meta[li][0]), int(meta[li][1])
        s = st[li, :grid].astype(np.float64)
        t0 = s[:, 0].min()
        starts.append(t0)
        ends.append(s[:, 1 + 2 * (nph - 1)].max())
        print(f"\nlaunch {li}: {nph} phases, grid {grid}, duration {(ends[-1] - t0) / 1e3:.1f} us"
              + (f", gap since the previous chain launch ended {(t0 - ends[-2]) / 1e3:.1f} us (attention kernel + boundaries)" if li else ""))
        print("| phase | work ended: min / median / max (us) | barrier released: first / last CTA (us) | phase time (us) |")
        print("|---|---|---|---|")
        prev = 0.0
        for ph in range(nph):
            e = s[:, 1 + 2 * ph]
            cell = "-"
            nxt = (e.max() - t0) / 1e3
            if ph + 1 < nph:
                b = s[:, 2 + 2 * ph]
                cell = f"{(b.min() - t0) / 1e3:.1f} / {(b.max() - t0) / 1e3:.1f}"
                nxt = (b.max() - t0) / 1e3
            label = names.get(nph, [f"phase {i}" for i in range(nph)])[ph]
            print(f"| {label} | {(e.min() - t0) / 1e3:.1f} / {(np.median(e) - t0) / 1e3:.1f} / {(e.max() - t0) / 1e3:.1f} | {cell} | {nxt - prev:.1f} |")
            prev = nxt


# ---------------------------------------------------------------------------------------------- cfg5 sweep
def run_sweep(args):
    """BASELINE.json configs[4]: concurrent decodes x prefill length at the 7B shape.  Prints one markdown table row per
    grid point (step latency, packed tok/s, achieved HBM GB/s = algorithmic bytes / latency, tensor TFLOP/s, fraction
    of the point's roofline at the measured peaks).  Not the bench line; a report for profiles/."""
    import torch
    from . import binding, inputs as I
    torch.cuda.set_device(0)
    cfg = I.cfg_7b_layers(args.layers)
    hw = I.make_weights(cfg, 4, threads=max(4, os.cpu_count() or 8))
    W = binding.WeightsFP8(cfg, quantize_on_device(cfg, hw, torch, I)) if args.fp8 else binding.Weights(cfg, hw)
    wbytes = 1.0 if args.fp8 else 2.0
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
           [(n, p) for n in (0, 1, 3, 6, 10, 15) for p in (0, 128, 276, 512) if not (args.fp8 and n + p > 512)]
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
            wk = step_work(cfg, segs, 0, wbytes)
            roof = max(wk["bytes"] / (peaks["hbm_gbs"] * 1e9), wk["flops"] / (peaks["tf_sustained"] * 1e12)) * 1e3
            print(f"| {n_dec} | {p_len} | {wk['T']} | {ms:.3f} | {wk['T'] / ms * 1e3:.0f} | {wk['bytes'] / ms / 1e6:.0f} | "
                  f"{wk['flops'] / ms / 1e9:.0f} | {roof:.3f} | {roof / ms:.2f} |", flush=True)



def run_attention_units(args):
    """The tcgen05 attention units (attention_umma.cuh, af_debug_attention(2)) as the layer chain's last phase: (a) the
    units' %globaltimer stamps (af_debug_trace(2)) for the steady cfg3 step on a 3-layer slice, by CTA group - CTAs 0..31
    start with the 20-row query tile (276 keys), 32..63 with rows 128..255, 64..95 with rows 0..127, 96..147 with decode
    rows; (b) the steady cfg3 step at --layers layers, attention_kernel (mode 1) against the units (mode 2), alternating in
    one process, CUDA events over 40 steps each.  --own-kernel: the per-stage path (AF_WEIGHTS_FP16), where the units run
    as attention_umma_kernel - the command the ncu capture of that kernel uses."""
    import numpy as np
    import torch
    from . import binding, inputs as I
    torch.cuda.set_device(0)

    def make(layers):
        cfg = I.cfg_7b_layers(layers)
        W = binding.Weights(cfg, I.make_weights(cfg, SEED, threads=16), prepared="fp16" if args.own_kernel else True)
        ring = binding.Ring(cfg, R_REGIONS, CAPACITY, max_rows=288)
        e_dev = [I.make_embeds(cfg, SEED, t, L_P + K_STAGES - 1).cuda() for t in range(8)]
        tau = [0]

        def step():
            t = tau[0]
            ring.reset_slot(t % R_REGIONS, -1)
            segs = I.steady_schedule(t, L_P, K_STAGES, R_REGIONS)
            ring.packed_forward(W, e_dev[t % 8][:I.total_rows(segs)], segs)
            tau[0] = t + 1
        return step

    binding.attention_mode(2)
    step = make(3)
    for _ in range(12):
        step()
    torch.cuda.synchronize()
    binding.chain_trace(2)
    step()
    st, meta, n = binding.chain_trace_read()
    binding.chain_trace(0)
    names = ["phase start", "lists", "1st unit: loads issued", "first chunk / K landed", "all landed", "S done / scores", "row maximum",
             "P written / probabilities", "O done", "unit end", "2nd unit: loads issued", "K landed", "-", "scores", "maximum",
             "probabilities", "-", "unit end"]
    print("(a) stamps of worker thread 0, us after the phase's first CTA started, mean over the CTA group; launches:", n)
    for li in range(min(n, 2)):
        s = st[li, :int(meta[li][1])].astype(np.float64)
        t0 = s[:, 0][s[:, 0] > 0].min()
        print(f"\nlaunch {li}: last stamp {(s.max() - t0) / 1e3:.1f} us\n| stamp | CTAs 0-31 | CTAs 32-63 | CTAs 64-95 | CTAs 96-147 |\n|---|---|---|---|---|")
        for k in range(18):
            cells = []
            for lo, hi in ((0, 32), (32, 64), (64, 96), (96, 148)):
                col = s[lo:hi, k]
                col = col[col > 0]
                cells.append(f"{(col.mean() - t0) / 1e3:.1f}" if len(col) else "-")
            if names[k] != "-":
                print(f"| {names[k]} | " + " | ".join(cells) + " |")
    del step
    step = make(args.layers)
    for _ in range(K_STAGES + 10):
        step()
    res = {1: [], 2: []}
    for _ in range(4):
        for mode in (1, 2):
            binding.attention_mode(mode)
            for _ in range(5):
                step()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(40):
                step()
            e1.record()
            torch.cuda.synchronize()
            res[mode].append(e0.elapsed_time(e1) / 40)
    binding.attention_mode(0)
    print(f"\n(b) steady cfg3 step, {args.layers} layers, ms per step (no LM head), four alternating repetitions:")
    print("attention_kernel (mma.sync, own launches):", " ".join(f"{x:.3f}" for x in res[1]))
    print("tcgen05 units (last phase of the chain):  ", " ".join(f"{x:.3f}" for x in res[2]))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--layers", type=int, default=32)
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--chunks", action="store_true", help="with --sweep: K = 7, 16, 24, 32 (276-row prefill + K - 1 decodes)")
    ap.add_argument("--fp8", action="store_true", help="AF_WEIGHTS_FP8 instead of the 16-bit weights")
    ap.add_argument("--chain-timeline", action="store_true")
    ap.add_argument("--library-gemm", action="store_true")
    ap.add_argument("--attention-units", action="store_true")
    ap.add_argument("--own-kernel", action="store_true", help="with --attention-units: the per-stage path, units as attention_umma_kernel")
    args = ap.parse_args()
    if args.library_gemm:
        return run_library_gemm(args)
    if args.chain_timeline:
        return run_chain_timeline(args)
    if args.attention_units:
        return run_attention_units(args)
    return run_sweep(args)


if __name__ == "__main__":
    main()
