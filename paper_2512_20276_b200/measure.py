"""Measurement helpers shared by bench.py and the report module: the algorithmic work model of one packed step
(SURVEY.md 8(d) / DESIGN.md "Roofline"), the measured peaks, and an nvidia-smi clock sampler.  No method arithmetic."""
from __future__ import annotations

import json
import os
import subprocess
import threading

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

L_P, K_STAGES, R_REGIONS, CAPACITY = 276, 7, 8, 512      # cfg3: 256 patch + 20 prompt tokens, K = 7 action tokens
SEED = 2


def step_work(cfg, segs, n_logit_rows, weight_bytes_per_elem=2.0):
    """Algorithmic FLOPs and bytes of one step.  weight_bytes_per_elem: 2 for the 16-bit formats, 1 for AF_WEIGHTS_FP8
    (projection matrices only: the LM head and the gains stay 16-bit; the per-channel scales are counted)."""
    D, F, V, Lyr, H, hd = cfg.d_model, cfg.ffn, cfg.vocab, cfg.n_layers, cfg.n_heads, cfg.head_dim
    T = sum(s[3] for s in segs)
    p_layer = 4 * D * D + 3 * D * F
    sum_ctx_rows = sum(sum(range(s[2] + 1, s[2] + s[3] + 1)) for s in segs)       # sum over rows of (pos+1)
    sum_ctx_segs = sum(s[2] + s[3] for s in segs)
    gemm_flops = 2 * T * Lyr * p_layer + 2 * n_logit_rows * V * D
    attn_flops = 4 * D * Lyr * sum_ctx_rows
    kv_row = 2 * H * hd * 2
    scales = 0 if weight_bytes_per_elem == 2.0 else 4 * Lyr * (5 * D + 2 * F)
    w_bytes = weight_bytes_per_elem * Lyr * p_layer + scales + 2 * (2 * Lyr + 1) * D + (2 * V * D if n_logit_rows else 0)
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


def quantize_on_device(cfg, host_weights, torch, I):
    """inputs.quantize_weights_fp8's per-matrix recipe (inputs.fp8_quantize) run on the GPU copy of each matrix: same
    codes and scales, seconds instead of a minute of host time at the 7B shape.  Returns the dict WeightsFP8 takes."""
    out = {"layers": [], "g_final": host_weights["g_final"], "w_lm": host_weights["w_lm"]}
    for L in host_weights["layers"]:
        q = {}
        for name, t in L.items():
            q[name] = I.fp8_quantize(t.cuda()) if name in I._FP8_MATRICES else t
        out["layers"].append(q)
    return out
