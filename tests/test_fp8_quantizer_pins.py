"""Pins of the weight-only FP8 input preparation: the E4M3 decode table against the
format's closed form and the library cast, round trip of every representable value, round-to-nearest-even on hand
midpoints, saturation at +-448, the per-output-channel scale's closed form and the error bound of the dequantised
weights.  CPU only; the CUDA path consumes the same codes and scales (tests/test_gpu_fp8.py)."""
import math

import torch

from paper_2512_20276_b200 import inputs as I


def test_decode_table_closed_form_and_library_cast():
    codes = torch.arange(256, dtype=torch.uint8)
    got = I.fp8_decode(codes)
    lib = codes.view(torch.float8_e4m3fn).to(torch.float32)
    ok = ~torch.isnan(lib)
    assert int((~ok).sum()) == 2 and bool(torch.isnan(got[0x7F])) and bool(torch.isnan(got[0xFF]))
    assert torch.equal(got[ok], lib[ok])
    # hand values: 0x38 = 1.0, 0x39 = 1.125, 0x7E = 448 (largest finite), 0x01 = 2^-9 (smallest subnormal), 0x08 = 2^-6
    assert float(got[0x38]) == 1.0 and float(got[0x39]) == 1.125 and float(got[0x7E]) == 448.0
    assert float(got[0x01]) == 2.0 ** -9 and float(got[0x08]) == 2.0 ** -6 and float(got[0xB8]) == -1.0
    assert float(got[0x00]) == 0.0


def test_every_representable_value_round_trips():
    codes = torch.tensor([c for c in range(256) if (c & 0x7F) != 0x7F and c != 0x80], dtype=torch.uint8)
    vals = I.fp8_decode(codes)
    # one row per value, padded with the format maximum so that the row scale is exactly 1
    rows = torch.stack([vals, torch.full_like(vals, 448.0)], dim=1)
    q, s = I.fp8_quantize(rows)
    assert torch.equal(s, torch.ones_like(s))
    assert torch.equal(q[:, 0], codes) and bool((q[:, 1] == 0x7E).all())


def test_round_to_nearest_even_and_saturation():
    # midpoints between neighbours: 1.0625 (1.0 | 1.125) -> even mantissa 1.0; 1.1875 (1.125 | 1.25) -> 1.25;
    # 432 (416 | 448) -> 448 (mantissa 110 is even); 2^-10 (0 | 2^-9) -> 0
    row = torch.tensor([[1.0625, 1.1875, 432.0, 2.0 ** -10, 448.0, -447.9, 1.07, 0.0]])
    q, s = I.fp8_quantize(row)
    assert float(s[0]) == 1.0
    assert I.fp8_decode(q)[0].tolist() == [1.0, 1.25, 448.0, 0.0, 448.0, -448.0, 1.125, 0.0]
    # saturation: the row maximum maps to +-448 exactly and nothing becomes NaN, whatever the magnitude
    g = torch.Generator().manual_seed(3)
    w = torch.randn(64, 256, generator=g) * torch.logspace(-6, 6, 64)[:, None]
    q, s = I.fp8_quantize(w)
    d = I.fp8_decode(q)
    assert not bool(torch.isnan(d).any())
    assert torch.equal(d.abs().amax(dim=1), torch.full((64,), 448.0))


def test_scale_closed_form_and_error_bound():
    g = torch.Generator().manual_seed(4)
    w = (0.02 * torch.randn(96, 512, generator=g)).to(torch.bfloat16)
    q, s = I.fp8_quantize(w)
    assert torch.equal(s, w.float().abs().amax(dim=1) / 448.0)
    zero = torch.zeros(2, 16)
    qz, sz = I.fp8_quantize(zero)
    assert torch.equal(sz, torch.ones(2)) and int(qz.abs().max()) == 0
    deq = I.fp8_dequantize(q, s)
    # normals carry 3 mantissa bits: |err| <= 2^-4 |w| (half an ulp), subnormals (below 2^-6 of the scaled range): <= 2^-10 scale
    err = (deq - w.float()).abs()
    bound = torch.maximum(w.float().abs() * 2.0 ** -4, s[:, None] * 2.0 ** -10) * (1 + 1e-6)
    assert bool((err <= bound).all())
    rel = float(err.pow(2).sum().sqrt() / w.float().pow(2).sum().sqrt())
    assert 0.01 < rel < 0.04          # ~2.6 % RMS for Gaussian rows: the price of halving the weight bytes


def test_quantize_weights_dict_shapes_and_passthrough():
    cfg = I.CFG_TINY
    hw = I.make_weights(cfg, seed=0)
    qw = I.quantize_weights_fp8(hw)
    assert len(qw["layers"]) == cfg.n_layers and qw["dequant"]["w_lm"] is hw["w_lm"]
    for L, Q, Dq in zip(hw["layers"], qw["layers"], qw["dequant"]["layers"]):
        for name in ("wq", "wk", "wv", "wo", "w_gate", "w_up", "w_down"):
            codes, scale = Q[name]
            assert codes.dtype == torch.uint8 and codes.shape == L[name].shape and scale.shape == (L[name].shape[0],)
            assert torch.equal(Dq[name], I.fp8_decode(codes) * scale[:, None]) and Dq[name].dtype == torch.float32
        assert Q["g_attn"] is L["g_attn"] and Dq["g_mlp"] is L["g_mlp"]
