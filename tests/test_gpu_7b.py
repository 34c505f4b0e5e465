"""GPU parity at the full Llama-2-7B shapes of BASELINE.json configs[2..4], in the launch configuration bench.py times
(T = 282 packed rows, ring 8 x 512, PDL launches), against the unpacked fp32 CPU oracle.  Oracle cost bounds what
is compared: cfg3 compares pipeline steps 0..9 (fill, first steady steps, first region recycle) on every row; cfg5
compares all 63 non-empty points of the 16 x 4 grid against two oracle forwards (packing independence makes each
point a row selection); cfg4 runs the full wrap schedule (a) at 32 layers GPU-vs-GPU (wrapped bases vs all-zero
bases, bitwise, every step), (b) at 32 layers against the oracle for two of the eight requests through their whole
life (SURVEY.md 8(d)'s fallback: the oracle runs requests independently, so it steps only those two), and (c) on an
8-layer slice against the oracle for all eight requests.  Run with `pytest -m gpu` on a B200."""
import numpy as np
import pytest
import torch

from oracle import af_oracle as O
from paper_2512_20276_b200 import inputs as I
from af_harness import Pair, relmax, TOL

pytestmark = pytest.mark.gpu

L_P, K, R, C = 276, 7, 8, 512


@pytest.fixture(scope="module")
def binding():
    from paper_2512_20276_b200 import binding as b
    b.load_library()
    return b


@pytest.fixture(scope="module")
def w7b(binding):
    cfg = I.CFG_7B
    hw = I.make_weights(cfg, seed=2, threads=16)
    return cfg, hw, binding.Weights(cfg, hw)


def test_cfg3_pipeline_fill_steady_and_recycle(binding, w7b):
    """BASELINE.json configs[2]: schedule P9 (req = step mod 8, reset_slot before each prefill), steps 0..8: pipeline
    fill, steady steps with 6 decodes at contexts 277..282, and the first recycled regions at steps 8 and 9; logits on
    the prediction rows (row 275 + the decode rows) from the first steady step on.  The argmax (Alg. 1 l.5/l.8) must
    agree wherever the oracle's top-2 margin exceeds what the tolerance can flip (2 * TOL * max|ref|)."""
    cfg, hw, W = w7b
    P = Pair(cfg, hw, R=R, C=C, max_rows=288, oracle_dtype=torch.float32, dev_weights=W)
    worst_h, worst_l = 0.0, 0.0
    for t in range(10):
        P.reset(t % R, -1)
        segs = I.steady_schedule(t, L_P, K, R)
        e = I.make_embeds(cfg, 2, t, I.total_rows(segs))
        hid, ref = P.step(segs, e)
        worst_h = max(worst_h, relmax(hid, ref))
        if t >= K - 1:
            lg, ref_lg = P.check_logits(hid, ref, I.prediction_rows(segs))
            worst_l = max(worst_l, relmax(lg, ref_lg))
            top2 = ref_lg.topk(2, dim=1).values
            safe = (top2[:, 0] - top2[:, 1]) > 2 * TOL * ref_lg.abs().max()
            assert torch.equal(lg.argmax(dim=1).cpu()[safe], ref_lg.argmax(dim=1)[safe]), f"step {t}: argmax differs beyond the tolerance"
    for r in (8 % R, 9 % R):                                               # regions 0 and 1 were recycled and rotated
        assert P.base[r] == (L_P + K - 1) % C
    assert P.len[9 % R] == L_P and P.len[8 % R] == L_P + 1
    P.check_ring(list(range(R)), layers=[0, 15, 31])
    print(f"cfg3: worst hidden {worst_h:.3e}, worst logits {worst_l:.3e}")


def test_cfg3_steady_step_is_deterministic(binding, w7b):
    """Two runs of the same 8 steps give bit-identical hidden states and logits (order-fixed reductions)."""
    cfg, hw, W = w7b
    outs = []
    for _ in range(2):
        ring = binding.Ring(cfg, R, C, max_rows=288)
        for t in range(8):
            ring.reset_slot(t % R, -1)
            segs = I.steady_schedule(t, L_P, K, R)
            hid = ring.packed_forward(W, I.make_embeds(cfg, 2, t, I.total_rows(segs)).cuda(), segs)
        lg = ring.logits_rows(W, hid, I.prediction_rows(segs))
        outs.append((hid.clone(), lg.clone()))
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])


def test_cfg5_scheduling_shape_sweep(binding, w7b):
    """BASELINE.json configs[4]: n_dec in 0..15 x prefill in {0,128,276,512}; decode j's history is the first 276+j
    rows of one stream H, the prefill is the first P rows of one stream E.  The oracle runs E (512 rows) and H
    (291 rows) once; every grid point's rows are selections of those two results."""
    cfg, hw, W = w7b
    Rr, Cc = 17, 1024
    E = I.make_embeds(cfg, 4, 0, 512)
    H = I.make_embeds(cfg, 4, 1, 291)
    orc = O.Oracle(cfg, hw, torch.float32)
    ref_E = orc.step([(0, 0, 0, 512)], E)
    ref_H = orc.step([(1, 0, 0, 291)], H)
    ring = binding.Ring(cfg, Rr, Cc, max_rows=544)
    for j in range(15):                      # histories: region j+1 holds the first 276+j rows of H
        ring.packed_forward(W, H[:276 + j].cuda().contiguous(), [(j + 1, 0, 0, 276 + j)])
    assert ring.packed_forward(W, E[:0].cuda(), []).shape[0] == 0          # the (0, 0) grid point is a legal no-op
    worst = 0.0
    points = [(n, p) for n in range(16) for p in (0, 128, 276, 512)]          # the full 16 x 4 grid of configs[4]
    for n_dec, p_len in points:
        if n_dec == 0 and p_len == 0:
            continue
        ring.reset_slot(0, 0)
        for j in range(15):
            ring.set_len(j + 1, 276 + j)
        segs, rows, refs = [], [], []
        if p_len:
            segs.append((0, 0, 0, p_len)); rows.append(E[:p_len]); refs.append(ref_E[:p_len])
        for j in range(n_dec):
            segs.append((j + 1, 1, 276 + j, 1)); rows.append(H[276 + j:277 + j]); refs.append(ref_H[276 + j:277 + j])
        hid = ring.packed_forward(W, torch.cat(rows).cuda().contiguous(), segs)
        err = relmax(hid, torch.cat(refs))
        worst = max(worst, err)
        assert err <= TOL, f"n_dec={n_dec} prefill={p_len}: {err:.3e}"
    print(f"cfg5: worst hidden {worst:.3e} over {len(points) - 1} grid points")


def test_f2_longer_action_chunks(binding, w7b):
    """SURVEY.md 8(f) f2 (the paper's section 4.3 / Fig. 5 workload): K - 1 = 15, 23, 31 decode segments of K - 1
    different in-flight requests (contexts 277 .. 276 + K - 1) packed with one 276-row prefill, R = 33 regions.  Same
    oracle trick as cfg5: decode j's history is the first 276 + j rows of one stream H, so one 307-row oracle forward of
    H and one 276-row forward of E give every expected row."""
    cfg, hw, W = w7b
    max_dec = 31
    E = I.make_embeds(cfg, 6, 0, 276)
    H = I.make_embeds(cfg, 6, 1, 276 + max_dec)
    orc = O.Oracle(cfg, hw, torch.float32)
    ref_E = orc.step([(0, 0, 0, 276)], E)
    ref_H = orc.step([(1, 0, 0, 276 + max_dec)], H)
    ring = binding.Ring(cfg, max_dec + 2, 512, max_rows=320)
    for j in range(max_dec):
        ring.packed_forward(W, H[:276 + j].cuda().contiguous(), [(j + 1, 0, 0, 276 + j)])
    for n_dec in (15, 23, 31):
        ring.reset_slot(0, 0)
        for j in range(max_dec):
            ring.set_len(j + 1, 276 + j)
        segs = [(0, 0, 0, 276)] + [(j + 1, 1, 276 + j, 1) for j in range(n_dec)]
        x = torch.cat([E] + [H[276 + j:277 + j] for j in range(n_dec)])
        hid = ring.packed_forward(W, x.cuda().contiguous(), segs)
        ref = torch.cat([ref_E] + [ref_H[276 + j:277 + j] for j in range(n_dec)])
        err = relmax(hid, ref)
        print(f"f2: K = {n_dec + 1}: hidden {err:.3e}")
        assert err <= TOL, f"K={n_dec + 1}: {err:.3e}"


def _cfg4_schedule(rng, Cc, n_req):
    """Deterministic scheduler of BASELINE.json configs[3]: chunked prefills (U{128..512}, <= 4 chunks per step) until
    len = 1015, then one decode token per step up to len = 1023."""
    lens = [0] * n_req
    steps = []
    while any(n < Cc - 1 for n in lens):
        segs, chunks = [], 0
        for r in range(n_req):
            n = lens[r]
            if n >= Cc - 1:
                continue
            if n < 1015:
                if chunks == 4:
                    continue
                ln = int(min(rng.integers(128, 513), 1015 - n))
                segs.append((r, 0, n, ln)); chunks += 1
            else:
                ln = 1
                segs.append((r, 1, n, 1))
            lens[r] = n + ln
        steps.append(segs)
    return steps


@pytest.fixture(scope="module")
def w_cfg4():
    """BASELINE.json configs[3]: 32-layer 7B shape, seed 3 (host bf16 weights; the 8-layer slice test uses layers 0..7)."""
    return I.make_weights(I.cfg_7b_layers(32, vocab=512), seed=3, threads=16)


def _cfg4_inputs(Rr, Cc):
    rng = np.random.default_rng(3)
    bases = [int(Cc - rng.integers(1, 601)) for _ in range(Rr)]
    steps = _cfg4_schedule(np.random.default_rng(33), Cc, Rr)
    return bases, steps


def test_cfg4_wraparound_long_context_32_layers(binding, w_cfg4):
    """BASELINE.json configs[3] at its stated depth (32 layers, ring capacity 1024, 8 requests whose appends cross the
    wrap, prefill chunks U{128..512}, decodes up to context 1023).  Every step: the run with wrapped bases is
    bit-identical to the run with all bases 0 (wrap == linear, GPU-vs-GPU), and the rows of requests 1 and 6 match the
    fp32 oracle, which runs those two requests alone through their whole life (chunks across the wrap + decodes to
    1023); at the end their ring K/V, read in logical order (base + j) mod C, equals the oracle's linear cache."""
    cfg = I.cfg_7b_layers(32, vocab=512)
    W = binding.Weights(cfg, w_cfg4)
    Rr, Cc = 8, 1024
    bases, steps = _cfg4_inputs(Rr, Cc)
    watched = (1, 6)
    P = Pair(cfg, w_cfg4, R=Rr, C=Cc, max_rows=2048, bases=bases, oracle_dtype=torch.float32, dev_weights=W)
    ring0 = binding.Ring(cfg, Rr, Cc, max_rows=2048)
    worst = 0.0
    for t, segs in enumerate(steps):
        e = I.make_embeds(cfg, 3, t, I.total_rows(segs))
        hid, _ = P.step(segs, e, oracle=False)                      # bookkeeping and the row map are still checked bit-exactly
        hid0 = ring0.packed_forward(W, e.cuda(), segs)
        assert torch.equal(hid, hid0), f"step {t}: result depends on the ring rotation"
        r0 = 0
        for sg in segs:
            if sg[0] in watched:
                ref = P.orc.step([sg], e[r0:r0 + sg[3]])
                err = relmax(hid[r0:r0 + sg[3]], ref)
                worst = max(worst, err)
                assert err <= TOL, f"step {t}, request {sg[0]}: hidden {err:.3e}"
            r0 += sg[3]
    assert P.len == [Cc - 1] * Rr
    worst_kv = P.check_ring(list(watched), layers=[0, 15, 31])
    print(f"cfg4 (32 layers): {len(steps)} steps, worst hidden {worst:.3e}, worst ring K/V {worst_kv:.3e}")


def test_cfg4_wraparound_long_context(binding, w_cfg4):
    """BASELINE.json configs[3] on an 8-layer slice against the oracle for ALL eight requests (every request's appends
    cross its wrap, prefill chunks of 128..512 rows, decodes up to context 1023, ring read back in logical order), with
    the same bitwise base-invariance check."""
    cfg = I.cfg_7b_layers(8, vocab=512)
    hw = {"layers": w_cfg4["layers"][:8], "g_final": w_cfg4["g_final"], "w_lm": w_cfg4["w_lm"]}
    W = binding.Weights(cfg, hw)
    Rr, Cc = 8, 1024
    bases, steps = _cfg4_inputs(Rr, Cc)
    P = Pair(cfg, hw, R=Rr, C=Cc, max_rows=2048, bases=bases, oracle_dtype=torch.float32, dev_weights=W)
    ring0 = binding.Ring(cfg, Rr, Cc, max_rows=2048)
    worst = 0.0
    for t, segs in enumerate(steps):
        e = I.make_embeds(cfg, 3, t, I.total_rows(segs))
        hid, ref = P.step(segs, e)
        worst = max(worst, relmax(hid, ref))
        hid0 = ring0.packed_forward(W, e.cuda(), segs)
        assert torch.equal(hid, hid0), f"step {t}: result depends on the ring rotation"
    assert P.len == [Cc - 1] * Rr
    P.check_ring(list(range(Rr)))
    print(f"cfg4 (8-layer slice, all requests): {len(steps)} steps, worst hidden {worst:.3e}")
