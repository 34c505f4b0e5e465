#!/usr/bin/env python
"""bench.py — the steady-state pipelined step of BASELINE.json configs[2] on N B200s (replicas).

A "step" is one pass of the whole hot path over one packed batch: the 276-row
prefill of a new frame + 6 single-row decodes of the in-flight frames through the 32-layer Llama-2-7B-shaped stack,
then the LM head on the 7 prediction rows.  In steady state one step completes one action frame (7 action tokens).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

Prints ONE JSON line (see DESIGN.md "Measurement" for every field).  The report modes that used to live here (cfg5 sweep,
kernel timeline, cuBLAS context) are `python -m paper_2512_20276_b200.reports`.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2512_20276_b200.measure import (ClockSampler, L_P, K_STAGES, R_REGIONS, CAPACITY, SEED, load_peaks,  # noqa: E402
                                           quantize_on_device, step_work)

# DRAM bytes per layer_chain_kernel launch (dram__bytes_read.sum + dram__bytes_write.sum of the 7-phase launches of a steady
# step, ncu, cold caches): profiles/launches_r2.md.  Algorithmic weight bytes per launch: 404.8 MB (one layer).
CHAIN_TRAFFIC_BYTES_PER_LAUNCH = 426.8e6
WORKLOAD = "cfg3: 32-layer Llama-2-7B shape, steady pipelined step = 276-row prefill + 6 decodes (ctx 277..282) + LM head on 7 rows"


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


# ---------------------------------------------------------------------------------------------- our arm
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layers", type=int, default=32, help="debug only: fewer layers (the line then says so)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fp8", action="store_true", help="skip the fp8_weights extra leg (AF_WEIGHTS_FP8, SURVEY.md 8(f) f4)")
    ap.add_argument("--library-context", action="store_true", help="add roofline.library_same_shapes: cuBLAS on the step's four projection shapes, same run (context, ~1.5 s of library GEMMs; off by default so that the bench line runs only the product)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    import torch
    import torch.distributed as dist
    from paper_2512_20276_b200 import binding, inputs as I, replicas, reports

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
    # ---- one more step with the chain kernel's per-phase stamps on: where a whole-layer launch spends its time ----
    chain_phases = None
    if rank == 0:
        binding.chain_trace(True)
        step(e_dev[tau[0] % n_buf])
        torch.cuda.synchronize()
        st_, meta_, n_tr = binding.chain_trace_read()
        binding.chain_trace(False)
        full = [i for i in range(min(n_tr, 16)) if int(meta_[i][0]) == 7]       # whole-layer launches among the last 16
        if full:
            import numpy as np
            names = ["o_proj", "rows_mlp_norm", "gate_up_swiglu", "down_proj", "rows_attn_norm", "qkv_proj", "rope_append"]
            acc = np.zeros(7)
            for i in full:
                g_ = int(meta_[i][1])
                s_ = st_[i, :g_].astype(np.float64)
                t0_, prev_ = s_[:, 0].min(), 0.0
                for ph in range(7):
                    end_ = (s_[:, 2 + 2 * ph].max() if ph < 6 else s_[:, 1 + 2 * ph].max()) - t0_
                    acc[ph] += (end_ - prev_) / 1e3
                    prev_ = end_
            acc /= len(full)
            proj_us = float(acc[0] + acc[2] + acc[3] + acc[5])
            layer_flops = 2.0 * T * (4 * cfg.d_model ** 2 + 3 * cfg.d_model * cfg.ffn)
            chain_phases = {"what": "layer_chain_kernel, whole-layer launches of one step in this run (af_debug_trace, %globaltimer; "
                                    "a phase runs from the previous grid barrier's release to its own, max over the 148 CTAs)",
                            "launches": len(full), "us": {n_: float(v_) for n_, v_ in zip(names, acc)},
                            "launch_us": float(acc.sum()), "projection_phases_us": proj_us,
                            "projection_phases_tflops": layer_flops / proj_us / 1e6,
                            "projection_phases_weight_gbs": 2.0 * (4 * cfg.d_model ** 2 + 3 * cfg.d_model * cfg.ffn) / proj_us / 1e3}
    # ---- extra leg: the same steady step with AF_WEIGHTS_FP8 (E4M3 codes + per-output-channel scales,
    #      half the weight bytes in HBM); the headline stays the 16-bit line ----
    ms_fp8 = None
    if not args.no_fp8:
        W8 = binding.WeightsFP8(cfg, quantize_on_device(cfg, hw, torch, I))
        ring8 = binding.Ring(cfg, R_REGIONS, CAPACITY, max_rows=288)
        tau8 = [0]

        def step8(e):
            t = tau8[0]
            ring8.reset_slot(t % R_REGIONS, -1)
            segs = I.steady_schedule(t, L_P, K_STAGES, R_REGIONS)
            ring8.packed_forward(W8, e[:I.total_rows(segs)], segs, hidden_out=hidden)
            ring8.logits_rows(W8, hidden, I.prediction_rows(segs), logits_out=logits)
            tau8[0] = t + 1
        for _ in range(K_STAGES - 1 + max(3, warmup // 2)):
            step8(e_dev[tau8[0] % n_buf])
        barrier()
        ev8, ev9 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev8.record(stream)
        for _ in range(args.steps):
            step8(e_dev[tau8[0] % n_buf])
        ev9.record(stream)
        barrier()
        ms_fp8 = ev8.elapsed_time(ev9)
        del W8, ring8
    clocks = sampler.stop()

    ms_dev, ms_e2e, ms_loop, ms_graph, ms_fp8 = replicas.max_over_ranks([ms_dev, ms_e2e, ms_loop, ms_graph, ms_fp8 or 0.0], device="cuda")
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
                     "traffic": CHAIN_TRAFFIC_BYTES_PER_LAUNCH,
                     "peak_source": peaks["source"] + " sustained bf16 (kernel timed inside a long step)",
                     "launches_per_step": gemm_n, "avg_launch_ms": gemm_ms / max(1, gemm_n),
                     "share_of_step": gemm_ms / all_ms,
                     "weight_stream_gbs": work["weight_bytes"] / (gemm_ms / 1e3) / 1e9},
        "kernel_ms_per_step": {k: v[0] / n_prof for k, v in prof.items()},
        "chain_phases": chain_phases,
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
    if ms_fp8:
        wk8 = step_work(cfg, segs_steady, K_STAGES, 1.0)
        ms8 = ms_fp8 / args.steps
        roof8 = max(wk8["bytes"] / (peaks["hbm_gbs"] * 1e9), wk8["flops"] / (peaks["tf_sustained"] * 1e12)) * 1e3
        line["fp8_weights"] = {
            "what": "f4: the same steady step with AF_WEIGHTS_FP8 (E4M3 weight codes + per-output-channel fp32 scales streamed "
                    "from HBM, widened to fp16 in shared memory, fp16 activations, LM head 16-bit); same run, inputs resident",
            "value": replicas.whole_job_throughput(args.steps, ms_fp8), "unit": "frames/s", "ms_per_step": ms8,
            "weight_bytes": wk8["weight_bytes"], "bytes": wk8["bytes"],
            "step_roofline": {"ms_measured_peaks": roof8, "frac_of_measured": roof8 / ms8,
                              "bound": "tensor" if wk8["flops"] / (peaks["tf_sustained"] * 1e12) * 1e3 >= roof8 else "hbm"}}
    if world == 1 and args.layers == 32 and args.library_context:
        # context, not a product path: the vendor library's GEMMs on the same four shapes, timed the same way
        # (per-launch CUDA events, power-capped clock); see profiles/library_gemm_r1.md
        lib = reports.run_library_gemm(args, emit=False)
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
