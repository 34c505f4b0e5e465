"""The tcgen05 attention units (attention_umma.cuh; af_debug_attention(2)) against the oracle and against attention_kernel,
at the 7B head shape (32 heads x 128): as the layer chain's last phase (prepared gate|up weights), as the kernel of its own
(per-stage path), on the paper's steady schedule with wrapped ring bases, on ragged multi-segment steps (chunked prefills
with a prior context, 2-row and > 128-row segments, decode rows), and the automatic fall-back beyond 352 positions."""
import numpy as np
import pytest
import torch

from paper_2512_20276_b200 import inputs as I
from af_harness import Pair, relmax, TOL

pytestmark = pytest.mark.gpu

L_P, K, R, C = 276, 7, 8, 512


@pytest.fixture(scope="module")
def binding():
    from paper_2512_20276_b200 import binding as b
    b.load_library()
    yield b
    b.attention_mode(0)


@pytest.fixture(scope="module")
def w2(binding):
    cfg = I.cfg_7b_layers(2, vocab=512)
    return cfg, I.make_weights(cfg, seed=5, threads=16)


def _steady(P, cfg, n_steps, seed):
    hid = ref = None
    outs = []
    for t in range(n_steps):
        P.reset(t % R, -1)
        segs = I.steady_schedule(t, L_P, K, R)
        hid, ref = P.step(segs, I.make_embeds(cfg, seed, t, I.total_rows(segs)))
        outs.append(hid.clone())
    return outs


@pytest.mark.parametrize("prepared", [True, "fp16"])
def test_steady_schedule_wrapped_bases_vs_oracle_and_vs_mma_sync(binding, w2, prepared):
    """P9's schedule (276-row prefill + up to 6 decode rows at contexts 277..282) for 10 steps - fill, steady, first
    recycled regions - on bases that make every request wrap; every step against the fp32 oracle (TOL), the ring read
    back in logical order, and the whole run against attention_kernel (two correct kernels: agreement to rounding)."""
    cfg, hw = w2
    bases = [(r * 97 + 300) % C for r in range(R)]
    W = binding.Weights(cfg, hw, prepared=prepared)
    runs = {}
    for mode in (2, 1):
        binding.attention_mode(mode)
        P = Pair(cfg, hw, R=R, C=C, max_rows=288, bases=bases, oracle_dtype=torch.float32, dev_weights=W)
        if mode == 2:
            runs[mode] = _steady(P, cfg, 10, seed=5)
            P.check_ring(list(range(R)))
        else:
            runs[mode] = []
            for t in range(10):
                P.reset(t % R, -1)
                segs = I.steady_schedule(t, L_P, K, R)
                hid, _ = P.step(segs, I.make_embeds(cfg, 5, t, I.total_rows(segs)), oracle=False)
                runs[mode].append(hid.clone())
    worst = max(relmax(a, b) for a, b in zip(runs[2], runs[1]))
    assert worst <= 2e-3, f"tcgen05 units vs mma.sync kernel: {worst:.3e}"


def test_ragged_segments_with_prior_context(binding):
    """Unit lists beyond the paper's schedule: several multi-row segments per step, some continuing a request (start_pos >
    0), lengths 2 / 17 / 129 / 200 (two query tiles, the second ragged), decode rows in between, contexts up to 352 (the
    units' limit), random bases.  One 7B-shaped layer against the fp32 oracle."""
    cfg = I.CFG_7B_1L
    hw = I.make_weights(cfg, seed=9)
    rng = np.random.default_rng(9)
    binding.attention_mode(2)
    P = Pair(cfg, hw, R=6, C=384, max_rows=400, bases=[int(rng.integers(0, 384)) for _ in range(6)], oracle_dtype=torch.float32)
    steps = [
        [(0, 0, 0, 200), (1, 0, 0, 2), (2, 0, 0, 129), (3, 0, 0, 17)],
        [(0, 0, 200, 150), (1, 1, 2, 1), (2, 1, 129, 1), (3, 0, 17, 100), (4, 0, 0, 1)],       # request 0 reaches 350
        [(0, 1, 350, 1), (0 + 5, 0, 0, 31), (1, 0, 3, 128), (2, 1, 130, 1), (4, 1, 1, 1)],
        [(0, 1, 351, 1), (5, 1, 31, 1), (1, 1, 131, 1), (3, 0, 117, 2)],                       # context 352: the limit
    ]
    for t, segs in enumerate(steps):
        rows = sum(s[3] for s in segs)
        P.step(segs, I.make_embeds(cfg, 9, t, rows))
    P.check_ring(list(range(6)))


def test_contexts_beyond_the_units_fall_back_to_the_mma_sync_kernel(binding):
    """A 400-row prefill exceeds a unit's 352 positions: mode 2 must take attention_kernel for that step - bit-identical
    to mode 1 - and return to the units on the next eligible step."""
    cfg = I.CFG_7B_1L
    hw = I.make_weights(cfg, seed=4)
    W = binding.Weights(cfg, hw)
    e = I.make_embeds(cfg, 4, 0, 400).cuda()
    outs = []
    for mode in (1, 2):
        binding.attention_mode(mode)
        ring = binding.Ring(cfg, 2, 512, max_rows=512)
        outs.append(ring.packed_forward(W, e, [(0, 0, 0, 400)]).clone())
    assert torch.equal(outs[0], outs[1])


def test_units_are_deterministic(binding, w2):
    """Units are handed out dynamically; which CTA runs a unit must not change a bit of the result."""
    cfg, hw = w2
    W = binding.Weights(cfg, hw)
    binding.attention_mode(2)
    outs = []
    for rep in range(3):
        ring = binding.Ring(cfg, R, C, max_rows=288)
        for t in range(8):
            ring.reset_slot(t % R, -1)
            segs = I.steady_schedule(t, L_P, K, R)
            hid = ring.packed_forward(W, I.make_embeds(cfg, 5, t, I.total_rows(segs)).cuda(), segs)
        outs.append(hid.clone())
    assert torch.equal(outs[0], outs[1]) and torch.equal(outs[0], outs[2])


def test_default_mode_takes_the_units_for_decode_only_steps(binding):
    """Mode 0 (the default): a step made of one-row segments only runs the units as the chain's last phase - one launch
    fewer per layer than with attention_kernel - and a step with a multi-row segment does not.  Decode-only steps at contexts
    100..105 and 300..305 against the fp32 oracle, ring checked."""
    cfg = I.CFG_7B_1L
    hw = I.make_weights(cfg, seed=6)
    binding.attention_mode(0)
    P = Pair(cfg, hw, R=4, C=384, max_rows=400, bases=[380, 17, 200, 0], oracle_dtype=torch.float32)
    n0 = binding.launch_count()
    P.step([(0, 0, 0, 100), (1, 0, 0, 300)], I.make_embeds(cfg, 6, 0, 400))
    prefill_launches = binding.launch_count() - n0
    for t in range(6):
        n0 = binding.launch_count()
        P.step([(0, 1, 100 + t, 1), (1, 1, 300 + t, 1)], I.make_embeds(cfg, 6, 1 + t, 2))
        assert binding.launch_count() - n0 == prefill_launches - cfg.n_layers
    P.check_ring([0, 1])


def test_random_schedules_units_vs_mma_sync(binding):
    """150 random packed steps on one 7B-shaped layer - requests appear, grow by chunks of 1..180 rows or by single decode
    rows, and are recycled at random bases before they pass 352 positions - run twice, with the units (mode 2) and with
    attention_kernel (mode 1).  Every step's hidden states agree to rounding; the units' unit lists, look-ahead loads,
    dynamic hand-out and wrap handling see shapes no fixed schedule has."""
    cfg = I.CFG_7B_1L
    hw = I.make_weights(cfg, seed=12)
    W = binding.Weights(cfg, hw)
    Rr, Cc, LIM = 8, 400, 352
    worst = 0.0
    outs = {}
    for mode in (2, 1):
        binding.attention_mode(mode)
        rng = np.random.default_rng(123)
        ring = binding.Ring(cfg, Rr, Cc, max_rows=512)
        length = [0] * Rr
        outs[mode] = []
        for t in range(150):
            segs, rows = [], 0
            for r in rng.permutation(Rr):
                r = int(r)
                if length[r] >= LIM - 1 or (length[r] > 0 and rng.random() < 0.05):
                    ring.reset_slot(r, int(rng.integers(0, Cc)))
                    length[r] = 0
                    continue
                kind = rng.random()
                if kind < 0.35:
                    continue
                ln = 1 if (kind < 0.7 and length[r] > 0) else int(min(rng.integers(1, 181), LIM - length[r]))
                if rows + ln > 512:
                    continue
                segs.append((r, 1 if (ln == 1 and length[r] > 0) else 0, length[r], ln))
                length[r] += ln
                rows += ln
            if not segs:
                continue
            hid = ring.packed_forward(W, I.make_embeds(cfg, 12, t, rows).cuda(), segs)
            outs[mode].append(hid.clone())
    assert len(outs[1]) == len(outs[2]) and len(outs[1]) > 100
    for a, b in zip(outs[2], outs[1]):
        assert not torch.isnan(a).any()
        worst = max(worst, relmax(a, b))
    assert worst <= 2e-3, f"units vs attention_kernel over random schedules: {worst:.3e}"


def test_units_on_a_two_chunk_step(binding):
    """A packed step of 800 rows (eight 100-row prefills) runs the layer chain with two token chunks per weight tile; its
    last phase is still the attention units (256 tensor units on 148 CTAs: every CTA takes two).  Then 8 decode rows."""
    cfg = I.CFG_7B_1L
    hw = I.make_weights(cfg, seed=8)
    binding.attention_mode(2)
    P = Pair(cfg, hw, R=8, C=256, max_rows=1024, bases=[250, 0, 13, 100, 255, 77, 200, 31], oracle_dtype=torch.float32)
    P.step([(r, 0, 0, 100) for r in range(8)], I.make_embeds(cfg, 8, 0, 800))
    P.step([(r, 1, 100, 1) for r in range(8)], I.make_embeds(cfg, 8, 1, 8))
    P.check_ring(list(range(8)))


def test_units_with_fp8_weights(binding):
    """AF_WEIGHTS_FP8 runs on the layer chain only, so with mode 2 its attention is the chain's last phase too
    (layer_chain_kernel<true, *>): the steady schedule's first 8 steps, units against attention_kernel, same weights."""
    cfg = I.cfg_7b_layers(2, vocab=512)
    W = binding.WeightsFP8(cfg, I.quantize_weights_fp8(I.make_weights(cfg, seed=5, threads=16)))
    outs = {}
    for mode in (2, 1):
        binding.attention_mode(mode)
        ring = binding.Ring(cfg, R, C, max_rows=288)
        for r in range(R):
            ring.reset_slot(r, (r * 131 + 290) % C)
        outs[mode] = []
        for t in range(8):
            ring.reset_slot(t % R, -1)
            segs = I.steady_schedule(t, L_P, K, R)
            outs[mode].append(ring.packed_forward(W, I.make_embeds(cfg, 5, t, I.total_rows(segs)).cuda(), segs).clone())
    worst = max(relmax(a, b) for a, b in zip(outs[2], outs[1]))
    assert worst <= 2e-3, f"FP8 weights, units vs attention_kernel: {worst:.3e}"
