"""f1: Algorithm 1's pipeline loop with its state on the device (af_loop_*), through the C ABI.

What is unique is compared exactly, what floating point decides is compared in the precision that decided it:
  * the device-side segment table / ring bookkeeping against the oracle's integer index model, bit-exact, every step;
  * the graph-replayed loop against the same steps driven from the host through af_packed_forward / af_logits_rows /
    af_argmax_rows / af_embed_rows on a second ring: bit-identical logits and tokens (the kernels are deterministic);
  * every token is the oracle's argmax definition applied to the library's own fp32 logits;
  * every completed frame against oracle.greedy_frame (the frame run alone, unpacked), teacher-forced along the
    library's tokens: logits within the north-star tolerance, and the oracle's own token wherever its top-2 margin
    exceeds what that tolerance can flip.
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


def _table(cfg, seed):
    g = torch.Generator().manual_seed(seed)
    return torch.randn(cfg.vocab, cfg.d_model, generator=g).to(torch.bfloat16)


@pytest.mark.parametrize("use_graph", [True, False])
def test_device_loop_tiny(binding, use_graph):
    cfg, R, C, L_P, K, n_steps = I.CFG_TINY, 5, 128, 40, 4, 14
    hw = I.make_weights(cfg, seed=0)
    W = binding.Weights(cfg, hw)
    table = _table(cfg, 41)
    table_d = table.cuda()
    frames = [I.make_embeds(cfg, 41, t, L_P) for t in range(n_steps)]
    bases = [100, 0, 127, 60, 90]                       # appends cross the wrap in several regions

    ring = binding.Ring(cfg, R, C, max_rows=128)
    host = binding.Ring(cfg, R, C, max_rows=128)         # the same steps, driven from the host
    for r, b in enumerate(bases):
        ring.reset_slot(r, b)
        host.reset_slot(r, b)
    loop = binding.Loop(W, ring, table_d, L_P, K)
    st = torch.cuda.Stream()
    base, length = list(bases), [0] * R
    got_tok, got_lg, frames_out = [], [], {}
    prev_host_tok = None
    for t in range(n_steps):
        segs = I.steady_schedule(t, L_P, K, R)
        n_dec = len(segs) - 1
        with torch.cuda.stream(st):
            loop.prefill_embeds.copy_(frames[t].cuda(), non_blocking=False)
            loop.step(use_graph=use_graph, stream=st)
        st.synchronize()
        assert loop.steps_done == t + 1
        # ---- integer state: device table == index model, bit-exact
        base[t % R], length[t % R] = O.ring_reset_model(C, base[t % R], length[t % R], -1)
        mr, mp, ms, length = O.ring_index_model(R, C, base, length, segs)
        assert ring.row_map(len(mr)) == (mr, mp, ms), f"step {t}: device row map differs from the index model"
        for r in range(R):
            assert ring.get_state(r) == (base[r], length[r])
        tok = loop.tokens[:1 + n_dec].cpu().tolist()
        lg = loop.logits[:1 + n_dec].cpu()
        assert tok == O.argmax_rows(lg), f"step {t}: token is not the lowest-index maximum of the library's logits"
        got_tok.append(tok); got_lg.append(lg)
        fr = loop.frame.cpu().tolist()
        if t >= K - 1:
            assert fr[0] == t - (K - 1)
            frames_out[fr[0]] = fr[1:]
        else:
            assert fr[0] == -1
        # ---- the same step through the host-driven public calls: bit-identical
        host.reset_slot(t % R, -1)
        emb = frames[t].cuda()
        if n_dec:
            emb = torch.cat([emb, binding.embed_rows(table_d, prev_host_tok[:n_dec])])
        hid = host.packed_forward(W, emb, segs)
        hlg = host.logits_rows(W, hid, I.prediction_rows(segs))
        prev_host_tok = binding.argmax_rows(hlg)
        assert torch.equal(hlg.cpu(), lg), f"step {t}: loop logits differ from the host-driven step"
        assert prev_host_tok.cpu().tolist() == tok
        assert torch.equal(loop.hidden[:L_P + n_dec].cpu(), hid.cpu())

    # ---- completed frames against the frame run alone by the oracle (A_sequences, Alg. 1 l.9)
    orc = O.Oracle(cfg, hw, torch.float64)
    assert sorted(frames_out) == list(range(n_steps - K + 1))
    n_margin = 0
    for f, toks in frames_out.items():
        assert toks == [got_tok[f + s][s] for s in range(K)], "A_sequences differs from the per-step tokens"
        own, ref = O.greedy_frame(orc, 0, frames[f], table, K, forced=toks)
        for s in range(K):
            lg = got_lg[f + s][s].double()
            assert relmax(lg, ref[s]) <= TOL, (f, s)
            top2 = torch.topk(ref[s], 2).values
            if float(top2[0] - top2[1]) > 2 * TOL * float(ref[s].abs().max()):
                assert toks[s] == own[s], (f, s)
                n_margin += 1
    assert n_margin > 0
    loop.destroy()


def test_loop_create_rejects_bad_geometry(binding):
    cfg = I.CFG_TINY
    W = binding.Weights(cfg, I.make_weights(cfg, seed=0))
    table = _table(cfg, 1).cuda()
    ring = binding.Ring(cfg, 4, 128, max_rows=128)
    with pytest.raises(binding.AfError):
        binding.Loop(W, ring, table, 40, 5)               # K > R
    with pytest.raises(binding.AfError):
        binding.Loop(W, ring, table, 126, 4)              # L_P + K - 1 > C
    binding.Loop(W, ring, table, 125, 4).destroy()        # exactly fills a region


# ------------------------------------------------------------------------------------------------ f3: sliding window
@pytest.mark.parametrize("W", [128, 40, 1])
def test_f3_sliding_window_tiny(binding, W):
    """A request outgrows its region: appends overwrite the oldest slots, rows attend the last W positions.  The oracle
    keeps a linear unbounded cache and a banded mask ("wrap == linear window").  Covers W = C (decode-only sliding),
    W < C with wrapping prefill chunks of the largest legal length C - W + 1, W = 1, rejected segments, and the
    live C positions of the ring against the oracle's cache."""
    from af_harness import Pair
    cfg, R, C, max_pos = I.CFG_TINY, 3, 128, 400
    hw = I.make_weights(cfg, seed=0)
    P = Pair(cfg, hw, R, C, max_rows=3 * C, bases=[100, 0, 77], window=W, max_pos=max_pos)
    big = C - W + 1                                        # largest chunk that may wrap
    pos = [0, 0, 0]
    step = [0]

    def run(segs):
        T = sum(s[3] for s in segs)
        hid, ref = P.step(segs, I.make_embeds(cfg, 6, step[0], T))
        step[0] += 1
        for s in segs:
            pos[s[0]] += s[3]
        return hid, ref

    run([(0, 0, 0, 100), (1, 0, 0, 128), (2, 0, 0, 60)])                   # inside the regions: v1 behaviour (+ window)
    # request 1 is full: one more token is legal only through the window rule
    for _ in range(3):
        run([(0, 1, pos[0], 1), (1, 1, pos[1], 1), (2, 1, pos[2], 1)])
    if big > 1:                                                           # a wrapping chunk of the largest legal length
        n = min(big, 120)
        run([(0, 0, pos[0], n), (1, 1, pos[1], 1)])
        with pytest.raises(binding.AfError):                              # one row more than the rule allows
            P.ring.packed_forward(P.W, I.make_embeds(cfg, 6, 99, big + 1).cuda(), [(1, 0, pos[1], big + 1)])
    else:
        with pytest.raises(binding.AfError):                              # W = C: only single tokens may slide
            P.ring.packed_forward(P.W, I.make_embeds(cfg, 6, 99, 2).cuda(), [(1, 0, pos[1], 2)])
    for r in range(R):
        assert P.ring.get_state(r) == (P.base[r], P.len[r])               # a rejected step leaves the state unchanged
    hid = ref = None
    for _ in range(4):                                                    # keep sliding: decodes + small chunks
        segs = [(1, 1, pos[1], 1), (2, 0, pos[2], min(big, 33))]
        hid, ref = run(segs)
    assert pos[1] > C
    P.check_ring([0, 1, 2])
    P.check_logits(hid, ref, I.prediction_rows(segs))
    with pytest.raises(binding.AfError):                                  # positions stay below max_pos
        P.ring.set_len(1, max_pos - 1)
        P.ring.packed_forward(P.W, I.make_embeds(cfg, 6, 98, 2).cuda(), [(1, 0, max_pos - 1, 2)])


def test_f3_window_base_invariance_and_reset(binding):
    """Bitwise: the windowed path gives identical results for any base rotation (KV tiles are walked in logical order),
    and af_ring_set_window refuses a non-empty ring."""
    cfg, C, W = I.CFG_TINY, 128, 64
    W_dev = binding.Weights(cfg, I.make_weights(cfg, seed=0))
    outs = []
    for b in (0, 93):
        ring = binding.Ring(cfg, 2, C, max_rows=C)
        ring.set_window(W, 300)
        ring.reset_slot(0, b)
        p, hid = 0, None
        for i, n in enumerate((128, 1, 40, 1, 65, 1)):
            hid = ring.packed_forward(W_dev, I.make_embeds(cfg, 8, i, n).cuda(), [(0, 0 if n > 1 else 1, p, n)])
            p += n
        outs.append(hid.cpu())
        with pytest.raises(binding.AfError):
            ring.set_window(0, 0)
    assert torch.equal(outs[0], outs[1])


# ------------------------------------------------------------------------------------------------ 7B shapes (hd = 128)
def test_f3_sliding_window_single_7b_layer(binding):
    """f3 at the Llama-2-7B layer shape (hd = 128 instantiation of the windowed attention kernel), ring 4 x 512,
    W = 256: the paper's 276-row prefill, then the request keeps growing past the region by decodes and by wrapping
    chunks of the largest legal length (257), packed with a second request that stays inside its region; fp32 oracle."""
    from af_harness import Pair
    cfg, C, W = I.CFG_7B_1L, 512, 256
    hw = I.make_weights(cfg, seed=1)
    P = Pair(cfg, hw, R=4, C=C, max_rows=320, bases=[400, 0, 17, 511], oracle_dtype=torch.float32, window=W, max_pos=1200)
    P.step([(0, 0, 0, 276), (1, 0, 0, 40)], I.make_embeds(cfg, 3, 0, 316))
    P.step([(0, 0, 276, 230), (1, 1, 40, 1)], I.make_embeds(cfg, 3, 1, 231))           # ends at 506, inside the region
    P.step([(0, 0, 506, 257), (1, 1, 41, 1)], I.make_embeds(cfg, 3, 2, 258))           # wraps: len = C - W + 1
    P.step([(0, 1, 763, 1), (1, 1, 42, 1)], I.make_embeds(cfg, 3, 3, 2))
    segs = [(0, 0, 764, 130), (1, 1, 43, 1), (2, 0, 0, 100)]
    hid, ref = P.step(segs, I.make_embeds(cfg, 3, 4, 231))
    P.check_ring([0, 1, 2])
    P.check_logits(hid, ref, I.prediction_rows(segs))
    with pytest.raises(binding.AfError):
        P.ring.packed_forward(P.W, I.make_embeds(cfg, 3, 5, 258).cuda(), [(0, 0, 894, 258)])


def test_device_loop_7b_shape_equals_host_driven_steps(binding):
    """f1 at bench.py's launch configuration (8-layer slice of the 7B shape, L_P = 276, K = 7, ring 8 x 512, graph
    replay): pipeline fill, the captured step and 6 replays with a region recycle are bit-identical (hidden, logits,
    tokens, row map) to the same steps issued through the host-driven calls, whose parity against the oracle is
    tests/test_gpu_7b.py's subject."""
    cfg = I.cfg_7b_layers(8)
    L_P, K, R, C, n_steps = 276, 7, 8, 512, 14
    W = binding.Weights(cfg, I.make_weights(cfg, seed=2, threads=16))
    table = (0.5 * torch.randn(cfg.vocab, cfg.d_model, generator=torch.Generator().manual_seed(9))).to(torch.bfloat16).cuda()
    ring, host = binding.Ring(cfg, R, C, max_rows=288), binding.Ring(cfg, R, C, max_rows=288)
    loop = binding.Loop(W, ring, table, L_P, K)
    st = torch.cuda.Stream()
    base, length, prev = [0] * R, [0] * R, None
    for t in range(n_steps):
        segs = I.steady_schedule(t, L_P, K, R)
        n_dec = len(segs) - 1
        e = I.make_embeds(cfg, 2, t, L_P).cuda()
        with torch.cuda.stream(st):
            loop.prefill_embeds.copy_(e)
            loop.step(use_graph=True, stream=st)
        st.synchronize()
        base[t % R], length[t % R] = O.ring_reset_model(C, base[t % R], length[t % R], -1)
        mr, mp, ms, length = O.ring_index_model(R, C, base, length, segs)
        assert ring.row_map(len(mr)) == (mr, mp, ms)
        host.reset_slot(t % R, -1)
        emb = torch.cat([e, binding.embed_rows(table, prev[:n_dec])]) if n_dec else e
        hid = host.packed_forward(W, emb, segs)
        lg = host.logits_rows(W, hid, I.prediction_rows(segs))
        prev = binding.argmax_rows(lg)
        assert torch.equal(loop.hidden[:L_P + n_dec], hid), t
        assert torch.equal(loop.logits[:1 + n_dec], lg), t
        assert torch.equal(loop.tokens[:1 + n_dec], prev), t
        assert loop.tokens[:1 + n_dec].cpu().tolist() == O.argmax_rows(lg.cpu())
    fr = loop.frame.cpu().tolist()
    assert fr[0] == n_steps - K
    loop.destroy()


@pytest.mark.parametrize("K,R,L_P", [(1, 1, 128), (2, 2, 17), (5, 5, 1)])
def test_device_loop_edge_shapes(binding, K, R, L_P):
    """Degenerate pipelines: no decode stage at all (K = 1, a region that is filled exactly and recycled every step),
    as many stages as regions (every region recycled the step after its frame completes), one-row prefills.
    Tokens and logits bit-identical to the host-driven steps, device table == index model."""
    cfg, C, n_steps = I.CFG_TINY, 128, 9
    W = binding.Weights(cfg, I.make_weights(cfg, seed=0))
    table = _table(cfg, 43).cuda()
    ring, host = binding.Ring(cfg, R, C, max_rows=128), binding.Ring(cfg, R, C, max_rows=128)
    loop = binding.Loop(W, ring, table, L_P, K)
    st = torch.cuda.Stream()
    base, length, prev = [0] * R, [0] * R, None
    for t in range(n_steps):
        segs = I.steady_schedule(t, L_P, K, R)
        n_dec = len(segs) - 1
        e = I.make_embeds(cfg, 43, t, L_P).cuda()
        with torch.cuda.stream(st):
            loop.prefill_embeds.copy_(e)
            loop.step(use_graph=True, stream=st)
        st.synchronize()
        base[t % R], length[t % R] = O.ring_reset_model(C, base[t % R], length[t % R], -1)
        mr, mp, ms, length = O.ring_index_model(R, C, base, length, segs)
        assert ring.row_map(len(mr)) == (mr, mp, ms)
        host.reset_slot(t % R, -1)
        emb = torch.cat([e, binding.embed_rows(table, prev[:n_dec])]) if n_dec else e
        hid = host.packed_forward(W, emb, segs)
        lg = host.logits_rows(W, hid, I.prediction_rows(segs))
        prev = binding.argmax_rows(lg)
        assert torch.equal(loop.logits[:1 + n_dec], lg) and torch.equal(loop.tokens[:1 + n_dec], prev), t
        fr = loop.frame.cpu().tolist()
        assert fr[0] == (t - (K - 1) if t >= K - 1 else -1)
        if t >= K - 1:
            assert fr[K] == int(prev[K - 1])
    loop.destroy()
