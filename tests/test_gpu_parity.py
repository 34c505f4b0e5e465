"""GPU parity tests proper: the CUDA path, called through the C ABI, against the unpacked CPU oracle on the same
seeded inputs.  Bit-exact for bookkeeping (row map, base/len), max|err| <= 2e-2 * max|ref| for tensors
(BASELINE.json north_star).  Run with `pytest -m gpu` on a B200."""
import numpy as np
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


# ------------------------------------------------------------------------------------------------ GEMM kernel
@pytest.mark.parametrize("n_tok,n_out,k", [
    (1, 128, 64), (16, 128, 64), (7, 512, 4096), (66, 256, 688), (66, 688, 256), (128, 256, 256),
    (144, 384, 512), (282, 4096, 4096), (282, 1000, 11008), (288, 4096, 1024), (300, 640, 448), (527, 768, 4096),
    (15, 32000, 512),
])
def test_gemm_tcgen05_vs_fp64(binding, n_tok, n_out, k):
    """out = a w^T through the tcgen05/TMA stream-K kernel; odd shapes span several tiles, a ragged feature tail,
    a ragged k tail (688 = 10.75 k-blocks), both token halves and the multi-launch token chunking."""
    g = torch.Generator().manual_seed(n_tok * 7919 + n_out * 31 + k)
    a = torch.randn(n_tok, k, generator=g).to(torch.float16)
    w = (0.05 * torch.randn(n_out, k, generator=g)).to(torch.bfloat16)
    ref = a.double() @ w.double().T
    got = binding.debug_gemm(a.cuda(), w.cuda())
    torch.cuda.synchronize()
    err = relmax(got, ref)
    assert err <= 1e-5, f"GEMM {n_tok}x{n_out}x{k}: max|err|/max|ref| = {err:.3e}"


def test_gemm_deterministic(binding):
    g = torch.Generator().manual_seed(5)
    a = torch.randn(282, 4096, generator=g).to(torch.float16).cuda()
    w = (0.02 * torch.randn(4096, 4096, generator=g)).to(torch.bfloat16).cuda()
    o1 = binding.debug_gemm(a, w).clone()
    o2 = binding.debug_gemm(a, w)
    assert torch.equal(o1, o2), "stream-K reduction must be order-fixed (bitwise repeatable)"


# ------------------------------------------------------------------------------------------------ cfg1
CFG1_STEP = [(0, 0, 0, 64), (1, 1, 70, 1), (2, 1, 127, 1)]


def _cfg1_run(bases):
    cfg = I.CFG_TINY
    hw = I.make_weights(cfg, seed=0)
    P = Pair(cfg, hw, R=4, C=128, max_rows=128, bases=bases)
    P.step([(1, 0, 0, 70)], I.make_embeds(cfg, 0, 0, 70))
    P.step([(2, 0, 0, 127)], I.make_embeds(cfg, 0, 1, 127))
    e = I.make_embeds(cfg, 0, 2, 66)
    hid, ref = P.step(CFG1_STEP, e)
    P.check_ring([0, 1, 2])
    lg, _ = P.check_logits(hid, ref, [63, 64, 65])
    return P, hid, lg


def test_cfg1_tiny_packed_step(binding):
    """BASELINE.json configs[0] with all bases 0."""
    _cfg1_run([0, 0, 0, 0])


def test_cfg1_wrapped_bases_and_capacity_error(binding):
    """configs[0] with bases (0,100,1,77): B wraps at pos 28, C's append at pos 127 lands in slot 0; outputs equal
    the base-0 run bitwise (KV tiles are walked in logical order); a further append to C is AF_ERR_CAPACITY with
    the state unchanged; a recycled region behaves as a fresh one."""
    _, hid0, lg0 = _cfg1_run([0, 0, 0, 0])
    P, hid1, lg1 = _cfg1_run([0, 100, 1, 77])
    assert torch.equal(hid0, hid1) and torch.equal(lg0, lg1), "ring rotation changed the result"
    cfg = I.CFG_TINY
    before = [P.ring.get_state(r) for r in range(4)]
    with pytest.raises(binding.AfError) as ei:
        P.ring.packed_forward(P.W, I.make_embeds(cfg, 0, 3, 1).cuda(), [(2, 1, 128, 1)])
    assert ei.value.code == binding.AF_ERR_CAPACITY
    assert [P.ring.get_state(r) for r in range(4)] == before
    P.reset(2, -1)
    assert P.ring.get_state(2) == ((1 + 128) % 128, 0)
    e = I.make_embeds(cfg, 0, 4, 64)
    hid_recycled, _ = P.step([(2, 0, 0, 64)], e)
    fresh = Pair(cfg, I.make_weights(cfg, seed=0), R=4, C=128, max_rows=128)
    hid_fresh, _ = fresh.step([(2, 0, 0, 64)], e)
    assert torch.equal(hid_recycled, hid_fresh)


def test_packed_equals_sequential_on_gpu(binding):
    """GPU-vs-GPU: the packed step equals the same segments run one per step (the paper's losslessness claim,
    P:224), to well inside the oracle tolerance."""
    cfg = I.CFG_TINY
    hw = I.make_weights(cfg, seed=0)
    W = binding.Weights(cfg, hw)
    e_hist = [I.make_embeds(cfg, 0, 0, 70), I.make_embeds(cfg, 0, 1, 127)]
    e = I.make_embeds(cfg, 0, 2, 66).cuda()
    outs = []
    for packed in (True, False):
        ring = binding.Ring(cfg, 4, 128, max_rows=128)
        ring.packed_forward(W, e_hist[0].cuda(), [(1, 0, 0, 70)])
        ring.packed_forward(W, e_hist[1].cuda(), [(2, 0, 0, 127)])
        if packed:
            outs.append(ring.packed_forward(W, e, CFG1_STEP).clone())
        else:
            parts, r0 = [], 0
            for s in CFG1_STEP:
                parts.append(ring.packed_forward(W, e[r0:r0 + s[3]].contiguous(), [s]).clone())
                r0 += s[3]
            outs.append(torch.cat(parts))
    err = relmax(outs[0], outs[1])
    assert err <= 2e-3, f"packed vs sequential on GPU: {err:.3e}"


def test_validation_errors_leave_state_unchanged(binding):
    cfg = I.CFG_TINY
    W = binding.Weights(cfg, I.make_weights(cfg, seed=0))
    ring = binding.Ring(cfg, 4, 128, max_rows=128)
    e = I.make_embeds(cfg, 0, 0, 8).cuda()
    bad = [([(4, 0, 0, 8)], "AF_ERR_SEGMENT"), ([(0, 0, 0, 4), (0, 0, 4, 4)], "AF_ERR_SEGMENT"),
           ([(0, 1, 0, 2)], "AF_ERR_SEGMENT"), ([(0, 0, 3, 8)], "AF_ERR_POSITION"), ([(0, 0, 0, 0)], "AF_ERR_SEGMENT")]
    for segs, name in bad:
        with pytest.raises(binding.AfError) as ei:
            ring.packed_forward(W, e, segs)
        assert ei.value.name == name, (segs, ei.value.name)
        with pytest.raises(ValueError, match=name):
            O.ring_index_model(4, 128, [0] * 4, [0] * 4, segs)
        assert all(ring.get_state(r) == (0, 0) for r in range(4))
    assert ring.packed_forward(W, e, []).shape[0] == 0          # n_segs == 0 is a legal no-op


def test_chunked_prefill_and_mixed_steps_tiny(binding):
    """cfg4 in miniature (tiny model so the fp64 oracle is fast): chunked prefills crossing each region's wrap,
    mixed prefill+decode steps, a run of decode-only steps up to the last slot; ring read back in logical order."""
    cfg = I.CFG_TINY
    hw = I.make_weights(cfg, seed=3)
    rng = np.random.default_rng(3)
    R, C = 4, 128
    bases = [int(C - rng.integers(1, 100)) for _ in range(R)]
    P = Pair(cfg, hw, R=R, C=C, max_rows=128, bases=bases)
    step = 0
    while any(n < C for n in P.len):
        segs = []
        rows = 0
        for r in range(R):
            n = P.len[r]
            if n >= C:
                continue
            if n < C - 6:
                ln = int(min(rng.integers(5, 40), C - 6 - n))
                if rows + ln > 128:
                    continue
                segs.append((r, 0, n, ln)); rows += ln
            else:
                segs.append((r, 1, n, 1)); rows += 1
        hid, ref = P.step(segs, I.make_embeds(cfg, 3, step, rows))
        step += 1
    assert P.len == [C] * R
    P.check_ring(list(range(R)))
    P.check_logits(hid, ref, list(range(hid.shape[0])))


# ------------------------------------------------------------------------------------------------ cfg2
def test_cfg2_single_7b_layer(binding):
    """BASELINE.json configs[1]: one Llama-2-7B-shaped layer, 276-row prefill + 6 decodes at contexts 277..282,
    ring 8 x 512; fp32 oracle (north_star: "a plain fp32 CPU implementation")."""
    cfg = I.CFG_7B_1L
    hw = I.make_weights(cfg, seed=1)
    P = Pair(cfg, hw, R=8, C=512, max_rows=288, bases=[0, 500, 37, 236, 511, 1, 300, 0], oracle_dtype=torch.float32)
    for s in range(1, 7):
        P.step([(s, 0, 0, 275 + s)], I.make_embeds(cfg, 1, s, 275 + s))
    segs = [(0, 0, 0, 276)] + [(s, 1, 275 + s, 1) for s in range(1, 7)]
    hid, ref = P.step(segs, I.make_embeds(cfg, 1, 0, 282))
    P.check_ring(list(range(7)))
    P.check_logits(hid, ref, I.prediction_rows(segs))


def test_bf16_weight_path_equals_prepared_fp16_path(binding):
    """AF_WEIGHTS_BF16 (every weight tile converted bf16 -> fp16 in shared memory by the GEMM) and AF_WEIGHTS_FP16
    (matrices prepared once by af_convert_bf16_to_fp16) hold the same values and take the same per-stage kernels, so
    they agree bit for bit.  AF_WEIGHTS_FP16_GU (gate | up also interleaved once by af_prepare_gate_up; ffn = 688 leaves
    a ragged last tile) runs the layer chain, whose projections add their k-pieces in a different (fixed) order: same
    values, agreement to rounding (1e-3 of the tensor's maximum, 20x inside the oracle tolerance)."""
    cfg = I.CFG_TINY
    hw = I.make_weights(cfg, seed=0)
    e = I.make_embeds(cfg, 0, 7, 100).cuda()
    outs = []
    for prepared in (True, "fp16", False):
        W = binding.Weights(cfg, hw, prepared=prepared)
        ring = binding.Ring(cfg, 4, 128, max_rows=128)
        hid = ring.packed_forward(W, e, [(0, 0, 0, 60), (3, 0, 0, 40)])
        outs.append((hid.clone(), ring.logits_rows(W, hid, [59, 99]).clone()))
    assert torch.equal(outs[1][0], outs[2][0]) and torch.equal(outs[1][1], outs[2][1])
    assert relmax(outs[0][0], outs[1][0]) <= 1e-3 and relmax(outs[0][1], outs[1][1]) <= 1e-3
    w = (0.02 * torch.randn(256, 512)).to(torch.bfloat16).cuda()
    w16 = torch.empty(256, 512, dtype=torch.float16, device="cuda")
    L = binding.load_library()
    assert L.af_convert_bf16_to_fp16(w.data_ptr(), w16.data_ptr(), w.numel(), None) == 0
    torch.cuda.synchronize()
    big = w.float().abs() >= 2.0 ** -14
    assert torch.equal(w16.float()[big], w.float()[big])                   # exact in the fp16 normal range
    assert float((w16.float() - w.float()).abs().max()) <= 2.0 ** -25        # fp16 subnormals below it


def test_prepare_gate_up_layout(binding):
    """af_prepare_gate_up: row t*128 + q*32 + half*16 + i of the packed matrix = row 64t + 16q + i of gate (half 0) or
    up (half 1), converted to fp16; rows of features >= ffn are zero (ffn = 688 leaves a 48-feature last tile).
    Bit-exact (index work)."""
    F, D = 688, 256
    g = torch.Generator().manual_seed(11)
    gate = (0.05 * torch.randn(F, D, generator=g)).to(torch.bfloat16)
    up = (0.05 * torch.randn(F, D, generator=g)).to(torch.bfloat16)
    L = binding.load_library()
    rows = L.af_gate_up_rows(F)
    assert rows == 128 * ((F + 63) // 64)
    out = torch.full((rows, D), 7.0, dtype=torch.float16, device="cuda")
    assert L.af_prepare_gate_up(gate.cuda().data_ptr(), up.cuda().data_ptr(), out.data_ptr(), F, D, None) == 0
    torch.cuda.synchronize()
    ref = torch.zeros(rows, D, dtype=torch.float16)
    for r in range(rows):
        t, q, half, i = r >> 7, (r >> 5) & 3, (r >> 4) & 1, r & 15
        f = 64 * t + 16 * q + i
        if f < F:
            ref[r] = (up if half else gate)[f].to(torch.float16)
    assert torch.equal(out.cpu(), ref)


@pytest.mark.parametrize("n_prefill", [257, 300, 509, 513, 800, 1021, 1100])
def test_wide_packed_steps_tiny(binding, n_prefill):
    """Packed steps wider than one UMMA N (two accumulator halves: 257, 300, 512 rows), wider than the 512 TMEM columns
    (516 .. 1024 rows: the layer chain walks two token chunks per weight tile) and wider than that (1103 rows: the
    per-stage path, three GEMM launches per projection) on the tiny model, whose ffn = 688 leaves a ragged SwiGLU tile: a
    long prefill that wraps its region, packed with decode rows of three other requests."""
    cfg = I.CFG_TINY
    hw = I.make_weights(cfg, seed=5)
    R, C = 4, 1280
    P = Pair(cfg, hw, R=R, C=C, max_rows=1280, bases=[1200, 0, 17, 1279])
    for r in (1, 2, 3):
        P.step([(r, 0, 0, 20 + r)], I.make_embeds(cfg, 5, r, 20 + r))
    segs = [(0, 0, 0, n_prefill)] + [(r, 1, 20 + r, 1) for r in (1, 2, 3)]
    hid, ref = P.step(segs, I.make_embeds(cfg, 5, 9, n_prefill + 3))
    P.check_ring([0, 1, 2, 3])
    P.check_logits(hid, ref, I.prediction_rows(segs))


def test_argmax_rows_bit_exact(binding):
    """f1: af_argmax_rows against the oracle's scalar definition on the SAME fp32 logits (an integer decided by floating
    point: both sides decide on the stored fp32 values): random rows at vocab 32000 and 1001, planted ties (the lowest
    index must win, wherever the tie sits in the block's reduction tree), NaNs, constant rows."""
    g = torch.Generator().manual_seed(21)
    for n, V in ((7, 32000), (5, 1001), (3, 17)):
        lg = torch.randn(n, V, generator=g)
        lg[0, V // 3] = lg[0, V - 1] = lg[0].max() + 1.0             # a tie far apart
        if n > 1:
            lg[1, 5] = float("nan"); lg[1, 6] = lg[1, 300 % V] = 9.0   # NaN next to a tie
        if n > 2:
            lg[2] = -2.5                                              # constant row -> 0
        got = binding.argmax_rows(lg.cuda()).cpu().tolist()
        assert got == O.argmax_rows(lg), (n, V)
    allnan = torch.full((2, 64), float("nan"))
    assert binding.argmax_rows(allnan.cuda()).cpu().tolist() == O.argmax_rows(allnan) == [0, 0]


def test_embed_rows_bit_exact(binding):
    g = torch.Generator().manual_seed(22)
    table = torch.randn(512, 256, generator=g).to(torch.bfloat16)
    toks = [0, 511, 17, 17, 512, -3, 255]
    got = binding.embed_rows(table.cuda(), torch.tensor(toks, dtype=torch.int32).cuda()).cpu()
    assert torch.equal(got, O.embed_rows(table, toks))


def test_closed_loop_tokens_on_device(binding):
    """f1 wiring on the tiny model: logits rows of a packed step -> af_argmax_rows -> af_embed_rows gives the next
    step's decode rows without the logits leaving the device; tokens equal the oracle's argmax of the same logits."""
    cfg = I.CFG_TINY
    hw = I.make_weights(cfg, seed=0)
    W = binding.Weights(cfg, hw)
    ring = binding.Ring(cfg, 4, 128, max_rows=128)
    hid = ring.packed_forward(W, I.make_embeds(cfg, 0, 0, 40).cuda(), [(0, 0, 0, 30), (1, 0, 0, 10)])
    lg = ring.logits_rows(W, hid, [29, 39])
    tok = binding.argmax_rows(lg)
    assert tok.cpu().tolist() == O.argmax_rows(lg.cpu())
    table = hw["w_lm"].to(torch.bfloat16).cuda().contiguous()         # any [V, D] bf16 table serves as the embedding
    nxt = binding.embed_rows(table, tok)
    assert torch.equal(nxt.cpu(), O.embed_rows(table.cpu(), tok.cpu().tolist()))
    hid2 = ring.packed_forward(W, nxt, [(0, 1, 30, 1), (1, 1, 10, 1)])
    assert hid2.shape[0] == 2 and torch.isfinite(hid2).all()
