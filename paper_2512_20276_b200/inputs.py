"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic: it only draws random numbers, rounds them once to bf16
(RNE) and builds segment tables (plain integer bookkeeping of the paper's schedule).
The recipe is stated in DESIGN.md ("Input recipe") and follows SURVEY.md 8(d):

  rng = numpy.random.default_rng([seed, layer, slot])   one independent stream per tensor (parallel-safe)
  projection weights  0.02 * N(0,1)            -> bf16
  RMSNorm gains       1 + 0.02 * N(0,1)        -> bf16   (reading A17)
  embeddings, step t  default_rng([seed, 1000 + t]).standard_normal((T, D)) -> bf16  (stand-in for projected
                      ViT patch + prompt + action-token embeddings, BASELINE.json north_star)

Everything is returned as torch CPU tensors of dtype bfloat16 (the exact values both sides consume).
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, asdict

import numpy as np
import torch

PHASE_PREFILL = 0
PHASE_DECODE = 1


@dataclass(frozen=True)
class ModelCfg:
    d_model: int
    n_layers: int
    n_heads: int
    head_dim: int
    ffn: int
    vocab: int
    rms_eps: float = 1e-5
    rope_theta: float = 1e4

    def as_dict(self):
        return asdict(self)


# BASELINE.json configs[0]: tiny correctness model.
CFG_TINY = ModelCfg(d_model=256, n_layers=2, n_heads=4, head_dim=64, ffn=688, vocab=512)
# BASELINE.json configs[1]: one Llama-2-7B-shaped layer (vocab kept small: the LM head is not part of cfg2).
CFG_7B_1L = ModelCfg(d_model=4096, n_layers=1, n_heads=32, head_dim=128, ffn=11008, vocab=512)
# BASELINE.json configs[2..4]: full 32-layer Llama-2-7B-shaped backbone.
CFG_7B = ModelCfg(d_model=4096, n_layers=32, n_heads=32, head_dim=128, ffn=11008, vocab=32000)


def cfg_7b_layers(n_layers: int, vocab: int = 32000) -> ModelCfg:
    return ModelCfg(d_model=4096, n_layers=n_layers, n_heads=32, head_dim=128, ffn=11008, vocab=vocab)


_LAYER_TENSORS = ("wq", "wk", "wv", "wo", "w_gate", "w_up", "w_down", "g_attn", "g_mlp")


def _shape(cfg: ModelCfg, name: str):
    D, F, V = cfg.d_model, cfg.ffn, cfg.vocab
    return {
        "wq": (D, D), "wk": (D, D), "wv": (D, D), "wo": (D, D),
        "w_gate": (F, D), "w_up": (F, D), "w_down": (D, F),
        "g_attn": (D,), "g_mlp": (D,), "g_final": (D,), "w_lm": (V, D),
    }[name]


def _draw(seed: int, layer: int, slot: int, shape, gain: bool) -> torch.Tensor:
    rng = np.random.default_rng([seed, layer, slot])
    a = rng.standard_normal(shape, dtype=np.float32)
    a *= np.float32(0.02)
    if gain:
        a += np.float32(1.0)
    return torch.from_numpy(a).to(torch.bfloat16)


def make_weights(cfg: ModelCfg, seed: int, threads: int = 8) -> dict:
    """{'layers': [ {name: bf16 tensor} ... ], 'g_final': ..., 'w_lm': ...} — all torch CPU bf16."""
    jobs = []
    for l in range(cfg.n_layers):
        for s, name in enumerate(_LAYER_TENSORS):
            jobs.append((l, name, (seed, l, s, _shape(cfg, name), name.startswith("g_"))))
    jobs.append((-1, "g_final", (seed, cfg.n_layers, 0, _shape(cfg, "g_final"), True)))
    jobs.append((-1, "w_lm", (seed, cfg.n_layers, 1, _shape(cfg, "w_lm"), False)))
    with ThreadPoolExecutor(max_workers=max(1, threads)) as ex:
        outs = list(ex.map(lambda j: _draw(*j[2]), jobs))
    w = {"layers": [dict() for _ in range(cfg.n_layers)]}
    for (l, name, _), t in zip(jobs, outs):
        if l >= 0:
            w["layers"][l][name] = t
        else:
            w[name] = t
    return w


def make_embeds(cfg: ModelCfg, seed: int, step: int, n_rows: int) -> torch.Tensor:
    """bf16 [n_rows, d_model] N(0,1) embeddings of packed step `step` (or of any named stream id)."""
    rng = np.random.default_rng([seed, 1000 + step])
    a = rng.standard_normal((n_rows, cfg.d_model), dtype=np.float32)
    return torch.from_numpy(a).to(torch.bfloat16)


# ---------------------------------------------------------------------------------------------------------
# Segment tables (tuples (req_id, phase, start_pos, len)).  Integer bookkeeping only.
# ---------------------------------------------------------------------------------------------------------

def steady_schedule(step: int, L_P: int, K: int, R: int):
    """Segment table of computation batch `step` of the paper's K-stage pipeline: the prefill of the
    newest request packed with decode stage s of the request that entered s steps ago, s = 1..K-1.
    Stage-s decode token sits at 0-indexed position L_P + s - 1 (context L_P + s; A4).
    During pipeline fill (step < K-1) only the stages that exist are present.  Requests use region step mod R."""
    assert R >= K
    segs = [(step % R, PHASE_PREFILL, 0, L_P)]
    for s in range(1, K):
        if step - s >= 0:
            segs.append(((step - s) % R, PHASE_DECODE, L_P + s - 1, 1))
    return segs


def prediction_rows(segs):
    """Packed row that predicts the next token of each segment = its last row (A3)."""
    rows, r0 = [], 0
    for (_, _, _, n) in segs:
        rows.append(r0 + n - 1)
        r0 += n
    return rows


def total_rows(segs) -> int:
    return sum(s[3] for s in segs)


# ---------------------------------------------------------------------------------------------------------
# f4 ("orthogonal to ... quantization"): weight-only FP8 storage.  Input preparation,
# not part of the method: a projection matrix W [out, in] is stored as one E4M3 code per element plus one fp32 scale
# per OUTPUT channel, scale_f = max_k |W_fk| / 448 (1 for an all-zero row), code_fk = E4M3(round-to-nearest-even of
# W_fk / scale_f, clamped to +-448).  Both sides consume the SAME dequantised values  W'_fk = value(code_fk) * scale_f:
# the oracle as fp32 matrices (fp8_dequantize), the CUDA library as the codes and the scales (it widens the codes to
# fp16 exactly and applies the scale to the fp32 accumulator).  E4M3 ("fn"): 1 sign, 4 exponent (bias 7), 3 mantissa
# bits, no infinities, 0x7f / 0xff = NaN, largest finite 448, subnormals m/8 * 2^-6.
# ---------------------------------------------------------------------------------------------------------
FP8_MAX = 448.0
_FP8_MATRICES = ("wq", "wk", "wv", "wo", "w_gate", "w_up", "w_down")


def fp8_decode(codes: torch.Tensor) -> torch.Tensor:
    """uint8 E4M3 codes -> fp32 values, by the format's definition (not by a library cast)."""
    c = codes.to(torch.int32)
    sign = torch.where((c & 0x80) != 0, -1.0, 1.0).to(torch.float32)
    e = ((c >> 3) & 0xF).to(torch.float32)
    m = (c & 0x7).to(torch.float32)
    normal = torch.pow(torch.tensor(2.0), e - 7.0) * (1.0 + m / 8.0)
    sub = (m / 8.0) * 2.0 ** -6
    v = torch.where(e > 0, normal, sub)
    v = torch.where((c & 0x7F) == 0x7F, torch.tensor(float("nan")), v)
    return sign * v


def fp8_quantize(w: torch.Tensor):
    """[out, in] matrix (any float dtype) -> (codes uint8 [out, in], scale fp32 [out])."""
    wf = w.to(torch.float32)
    amax = wf.abs().amax(dim=1)
    scale = torch.where(amax > 0, amax / FP8_MAX, torch.ones_like(amax))
    q = (wf / scale[:, None]).clamp(-FP8_MAX, FP8_MAX)
    codes = q.to(torch.float8_e4m3fn).view(torch.uint8)       # round to nearest even (library primitive, pinned in tests)
    return codes.contiguous(), scale.contiguous()


def fp8_dequantize(codes: torch.Tensor, scale: torch.Tensor) -> torch.Tensor:
    """The values both sides compute with: fp32 value(code) * scale of the row."""
    return fp8_decode(codes) * scale[:, None]


def quantize_weights_fp8(weights: dict) -> dict:
    """{'layers': [{name: (codes, scale)} for the seven projection matrices + the bf16 gains], 'dequant': a weights dict
    in make_weights' shape whose projection matrices are the fp32 dequantised values (for the oracle); g_final / w_lm
    are passed through (the LM head stays 16-bit)."""
    out = {"layers": [], "dequant": {"layers": [], "g_final": weights["g_final"], "w_lm": weights["w_lm"]},
           "g_final": weights["g_final"], "w_lm": weights["w_lm"]}
    for L in weights["layers"]:
        q, d = {}, {}
        for name, t in L.items():
            if name in _FP8_MATRICES:
                codes, scale = fp8_quantize(t)
                q[name] = (codes, scale)
                d[name] = fp8_dequantize(codes, scale)
            else:
                q[name] = t
                d[name] = t
        out["layers"].append(q)
        out["dequant"]["layers"].append(d)
    return out
