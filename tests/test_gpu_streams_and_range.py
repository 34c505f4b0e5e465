"""Library-state and numeric-range checks on the GPU (VERDICT r1 "What's weak" 11, 12):
 - two rings driven from two CUDA streams without any host synchronisation between their calls: both match the oracle
   (stream-K flags and the chain's grid barrier are per stream, and the library orders steps of different streams of a
   device behind each other);
 - large-magnitude activations: values stored as fp16 saturate at +-65504 instead of becoming inf, and a model whose
   activations are large but inside the fp16 range still meets the oracle tolerance.
Run with `pytest -m gpu` on a B200."""
import pytest
import torch

from oracle import af_oracle as O
from paper_2512_20276_b200 import inputs as I
from af_harness import relmax, TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2512_20276_b200 import binding as b
    b.load_library()
    return b


def test_two_rings_on_two_streams(binding):
    cfg = I.CFG_TINY
    hw = I.make_weights(cfg, seed=0)
    W = binding.Weights(cfg, hw)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    rings = [binding.Ring(cfg, 4, 128, max_rows=128) for _ in range(2)]
    orcs = [O.Oracle(cfg, hw, torch.float64) for _ in range(2)]
    sched = [[(0, 0, 0, 60)], [(1, 0, 0, 33), (0, 1, 60, 1)], [(2, 0, 0, 100), (0, 1, 61, 1), (1, 1, 33, 1)], [(0, 1, 62, 1), (1, 1, 34, 1), (2, 1, 100, 1)]]
    embeds = [[I.make_embeds(cfg, 20 + r, t, I.total_rows(s)) for t, s in enumerate(sched)] for r in range(2)]
    dev = [[e.cuda() for e in er] for er in embeds]
    torch.cuda.synchronize()
    outs = [[], []]
    for t, segs in enumerate(sched):                       # interleave the two rings' steps, no host sync in between
        for r in (0, 1):
            with torch.cuda.stream(streams[r]):
                outs[r].append(rings[r].packed_forward(W, dev[r][t], segs, stream=streams[r]))
    torch.cuda.synchronize()
    for r in (0, 1):
        for t, segs in enumerate(sched):
            ref = orcs[r].step(segs, embeds[r][t])
            err = relmax(outs[r][t], ref)
            assert err <= TOL, f"ring {r} step {t}: {err:.3e}"
    # the same two schedules run one ring after the other give bit-identical results (order-fixed reductions)
    ring = binding.Ring(cfg, 4, 128, max_rows=128)
    for t, segs in enumerate(sched):
        assert torch.equal(ring.packed_forward(W, dev[0][t], segs), outs[0][t])


def _scaled(hw, names, factor):
    out = {"layers": [dict(L) for L in hw["layers"]], "g_final": hw["g_final"], "w_lm": hw["w_lm"]}
    for L in out["layers"]:
        for n in names:
            L[n] = (L[n].float() * factor).to(torch.bfloat16)
    return out


def test_large_activations_inside_fp16_range_meet_the_tolerance(binding):
    """gate / up scaled x24: the SwiGLU product reaches ~1e4 (fp16 tops out at 65504), down scaled back; q/k/v scaled x8."""
    cfg = I.CFG_TINY
    hw = _scaled(_scaled(_scaled(I.make_weights(cfg, seed=0), ("w_gate", "w_up"), 24.0), ("w_down",), 1.0 / 64.0), ("wq", "wk", "wv"), 8.0)
    W = binding.Weights(cfg, hw)
    ring = binding.Ring(cfg, 4, 128, max_rows=128)
    orc = O.Oracle(cfg, hw, torch.float64)
    e = I.make_embeds(cfg, 0, 9, 90)
    segs = [(0, 0, 0, 90)]
    hid = ring.packed_forward(W, e.cuda(), segs)
    ref = orc.step(segs, e)
    assert bool(torch.isfinite(hid).all())
    err = relmax(hid, ref)
    print(f"large activations: hidden {err:.3e}")
    assert err <= TOL


def test_out_of_range_activations_saturate_instead_of_overflowing(binding):
    """gate / up scaled x400: silu(gate) * up exceeds 65504 for many elements.  The fp16 stores saturate (af.h "fp16
    range"), so every output stays finite; the oracle is not the expectation here (the format cannot hold the values)."""
    cfg = I.CFG_TINY
    hw = _scaled(_scaled(I.make_weights(cfg, seed=0), ("w_gate", "w_up"), 400.0), ("w_down",), 1e-4)
    for prepared in (True, "fp16"):                         # the layer chain and the per-stage path
        W = binding.Weights(cfg, hw, prepared=prepared)
        ring = binding.Ring(cfg, 4, 128, max_rows=128)
        e = I.make_embeds(cfg, 0, 9, 70)
        hid = ring.packed_forward(W, e.cuda(), [(0, 0, 0, 70)])
        assert bool(torch.isfinite(hid).all()), f"prepared={prepared}: inf / NaN in the residual stream"
    orc = O.Oracle(cfg, hw, torch.float64)
    ref = orc.step([(0, 0, 0, 70)], e)                       # confirms the premise: the exact product leaves the fp16 range
    x = O.rmsnorm(e.double(), hw["layers"][0]["g_mlp"].double(), cfg.rms_eps)
    assert float((O.silu(x @ hw["layers"][0]["w_gate"].double().T) * (x @ hw["layers"][0]["w_up"].double().T)).abs().max()) > 65504.0
