"""f4: weight-only FP8 storage (AF_WEIGHTS_FP8) against the oracle.  The input generator quantises the
bf16 weights (inputs.quantize_weights_fp8, pinned in tests/test_fp8_quantizer_pins.py); the oracle runs on the fp32
DEQUANTISED matrices, the CUDA library on the codes and scales, so the tolerance stays BASELINE.json's 2e-2.
Run with `pytest -m gpu` on a B200."""
import pytest
import torch

from oracle import af_oracle as O
from paper_2512_20276_b200 import inputs as I
from af_harness import Pair, relmax, TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2512_20276_b200 import binding as b
    b.load_library()
    return b


def test_prepare_gate_up_fp8_layout(binding):
    """af_prepare_gate_up_fp8 is a byte permutation: row t*128 + q*32 + half*16 + i of the packed matrix = row 64t + 16q + i
    of gate (half 0) or up (half 1); rows of features >= ffn are zero codes.  Bit-exact."""
    F, D = 688, 256
    g = torch.Generator().manual_seed(12)
    gate = torch.randint(0, 256, (F, D), generator=g, dtype=torch.uint8)
    up = torch.randint(0, 256, (F, D), generator=g, dtype=torch.uint8)
    L = binding.load_library()
    rows = L.af_gate_up_rows(F)
    out = torch.full((rows, D), 7, dtype=torch.uint8, device="cuda")
    assert L.af_prepare_gate_up_fp8(gate.cuda().data_ptr(), up.cuda().data_ptr(), out.data_ptr(), F, D, None) == 0
    torch.cuda.synchronize()
    ref = torch.zeros(rows, D, dtype=torch.uint8)
    for r in range(rows):
        t, q, half, i = r >> 7, (r >> 5) & 3, (r >> 4) & 1, r & 15
        f = 64 * t + 16 * q + i
        if f < F:
            ref[r] = (up if half else gate)[f]
    assert torch.equal(out.cpu(), ref)


def test_fp8_cfg1_tiny_packed_step(binding):
    """BASELINE.json configs[0] with FP8 weights: histories, the packed step (prefill 64 + decodes at 70 and 127, wrapped
    bases), ring K/V and logits against the oracle on the dequantised weights; row map and (base, len) bit-exact."""
    cfg = I.CFG_TINY
    qw = I.quantize_weights_fp8(I.make_weights(cfg, seed=0))
    W = binding.WeightsFP8(cfg, qw)
    P = Pair(cfg, qw["dequant"], R=4, C=128, max_rows=128, bases=[0, 100, 1, 77], dev_weights=W)
    P.step([(1, 0, 0, 70)], I.make_embeds(cfg, 0, 0, 70))
    P.step([(2, 0, 0, 127)], I.make_embeds(cfg, 0, 1, 127))
    hid, ref = P.step([(0, 0, 0, 64), (1, 1, 70, 1), (2, 1, 127, 1)], I.make_embeds(cfg, 0, 2, 66))
    P.check_ring([0, 1, 2])
    P.check_logits(hid, ref, [63, 64, 65])
    print(f"fp8 cfg1: hidden {relmax(hid, ref):.3e}")


def test_fp8_cfg2_single_7b_layer(binding):
    """configs[1] with FP8 weights: one 7B-shaped layer, 276-row prefill + 6 decodes at contexts 277..282."""
    cfg = I.CFG_7B_1L
    qw = I.quantize_weights_fp8(I.make_weights(cfg, seed=1, threads=16))
    W = binding.WeightsFP8(cfg, qw)
    P = Pair(cfg, qw["dequant"], R=8, C=512, max_rows=288, oracle_dtype=torch.float32, dev_weights=W)
    for s in range(1, 7):
        P.step([(s, 0, 0, 275 + s)], I.make_embeds(cfg, 1, s, 275 + s))
    segs = [(0, 0, 0, 276)] + [(s, 1, 275 + s, 1) for s in range(1, 7)]
    hid, ref = P.step(segs, I.make_embeds(cfg, 1, 10, 282))
    P.check_ring(list(range(7)))
    print(f"fp8 cfg2: hidden {relmax(hid, ref):.3e}")


def test_fp8_cfg3_pipeline_steps(binding):
    """configs[2] with FP8 weights at full depth (32 layers): pipeline fill and the first steady steps (0..6), logits on
    the prediction rows of the first steady step."""
    cfg = I.CFG_7B
    qw = I.quantize_weights_fp8(I.make_weights(cfg, seed=2, threads=16))
    W = binding.WeightsFP8(cfg, qw)
    L_P, K, R, C = 276, 7, 8, 512
    P = Pair(cfg, qw["dequant"], R=R, C=C, max_rows=288, oracle_dtype=torch.float32, dev_weights=W)
    worst = 0.0
    for t in range(7):
        P.reset(t % R, -1)
        segs = I.steady_schedule(t, L_P, K, R)
        hid, ref = P.step(segs, I.make_embeds(cfg, 2, t, I.total_rows(segs)))
        worst = max(worst, relmax(hid, ref))
    lg, ref_lg = P.check_logits(hid, ref, I.prediction_rows(segs))
    print(f"fp8 cfg3: worst hidden {worst:.3e}, logits {relmax(lg, ref_lg):.3e}")


def test_fp8_single_7b_layer_is_deterministic(binding):
    """The widened weight tiles are handed from the epilogue warps (generic proxy) to the tensor core (async proxy) of the
    pair's leader: a hand-over that let an MMA read a tile too early would show up as run-to-run differences.  Twelve
    repetitions of the cfg2 step are bit-identical."""
    cfg = I.CFG_7B_1L
    qw = I.quantize_weights_fp8(I.make_weights(cfg, seed=1, threads=16))
    W = binding.WeightsFP8(cfg, qw)
    ring = binding.Ring(cfg, 8, 512, max_rows=288)
    for s in range(1, 7):
        ring.packed_forward(W, I.make_embeds(cfg, 1, s, 275 + s).cuda(), [(s, 0, 0, 275 + s)])
    segs = [(0, 0, 0, 276)] + [(s, 1, 275 + s, 1) for s in range(1, 7)]
    e = I.make_embeds(cfg, 1, 10, 282).cuda()
    first = None
    for rep in range(12):
        ring.reset_slot(0, 0)
        for s in range(1, 7):
            ring.set_len(s, 275 + s)
        hid = ring.packed_forward(W, e, segs).clone()
        if first is None:
            first = hid
        assert torch.equal(hid, first), f"repetition {rep} differs"


def test_fp8_two_token_chunks_tiny(binding):
    """512 < T <= 1024 runs the layer chain with two token chunks per projection (FP8 weights): 700 packed rows."""
    cfg = I.CFG_TINY
    qw = I.quantize_weights_fp8(I.make_weights(cfg, seed=0))
    W = binding.WeightsFP8(cfg, qw)
    P = Pair(cfg, qw["dequant"], R=3, C=1024, max_rows=1024, dev_weights=W)
    P.step([(1, 0, 0, 33)], I.make_embeds(cfg, 0, 0, 33))
    hid, ref = P.step([(0, 0, 0, 650), (1, 1, 33, 1), (2, 0, 0, 49)], I.make_embeds(cfg, 0, 1, 700))
    P.check_ring([0, 1, 2])
    print(f"fp8, 700 rows: hidden {relmax(hid, ref):.3e}")


def test_fp8_rejects_wide_steps(binding):
    cfg = I.CFG_TINY
    qw = I.quantize_weights_fp8(I.make_weights(cfg, seed=0))
    W = binding.WeightsFP8(cfg, qw)
    ring = binding.Ring(cfg, 2, 2048, max_rows=2048)
    with pytest.raises(binding.AfError) as ei:
        ring.packed_forward(W, I.make_embeds(cfg, 0, 0, 1100).cuda(), [(0, 0, 0, 1100)])
    assert ei.value.code == binding.AF_ERR_UNSUPPORTED
    assert ring.get_state(0) == (0, 0)
