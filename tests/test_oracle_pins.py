"""Pins of the oracle against what the paper and the mathematics fix. CPU only."""
import math
import os

import pytest
import torch

from oracle import af_oracle as O
from paper_2512_20276_b200 import inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden")
F64 = torch.float64

SMALL = I.ModelCfg(d_model=64, n_layers=2, n_heads=4, head_dim=16, ffn=80, vocab=40)


def relerr(a, b):
    return float((a - b).abs().max() / b.abs().max())


# ---------------------------------------------------------------- P1 brute-force recompute (cache + causal logic)
@pytest.mark.parametrize("cfg,n,m", [(SMALL, 23, 9), (I.CFG_TINY, 40, 33)])
def test_p1_incremental_equals_bruteforce(cfg, n, m):
    w = I.make_weights(cfg, seed=5)
    e = I.make_embeds(cfg, 5, 0, n)
    ref = O.brute_forward(cfg, w, e)                       # no cache, explicit n x n mask, fp64
    o = O.Oracle(cfg, w, F64)
    got = [o.step([(0, 0, 0, m)], e[:m])]                  # prefill m, then decode one by one
    for p in range(m, n):
        got.append(o.step([(0, 1, p, 1)], e[p:p + 1]))
    got = torch.cat(got)
    assert relerr(got, ref) < 1e-9
    # fp32 mode of the same oracle stays within fp32 rounding of the fp64 brute force
    o32 = O.Oracle(cfg, w, torch.float32)
    got32 = o32.step([(0, 0, 0, n)], e)
    assert relerr(got32.double(), ref) < 1e-4


# ---------------------------------------------------------------- P2 RMSNorm closed forms
def test_p2_rmsnorm_closed_forms():
    g = torch.tensor([1.0, 2.0, -1.0, 0.5], dtype=F64)
    x = torch.tensor([[3.0, 4.0, 0.0, 0.0]], dtype=F64)
    # mean(x^2) = 25/4 -> rms = 2.5 ; x/rms = (1.2, 1.6, 0, 0)
    assert torch.allclose(O.rmsnorm(x, g, 0.0), torch.tensor([[1.2, 3.2, 0.0, 0.0]], dtype=F64), atol=1e-15)
    c, eps = 0.7, 1e-5
    out = O.rmsnorm(torch.full((1, 4), c, dtype=F64), g, eps)
    assert torch.allclose(out, g * c / math.sqrt(c * c + eps), atol=1e-15)
    z = O.rmsnorm(torch.zeros(2, 4, dtype=F64), g, eps)
    assert torch.equal(z, torch.zeros(2, 4, dtype=F64))     # no NaN at x = 0
    # scale invariance up to eps: norm(a x) == norm(x) when eps = 0
    x = torch.randn(3, 8, dtype=F64)
    assert torch.allclose(O.rmsnorm(5 * x, torch.ones(8, dtype=F64), 0.0), O.rmsnorm(x, torch.ones(8, dtype=F64), 0.0))


# ---------------------------------------------------------------- P3 RoPE worked values + group properties
def test_p3_rope_worked_values_from_golden_file():
    n_cases = 0
    for line in open(os.path.join(GOLD, "rope_worked_values.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        head, vin, vout = [s.split() for s in line.split("|")]
        hd, theta, pos = int(head[0]), float(head[1]), int(head[2])
        t = torch.tensor([float(v) for v in vin], dtype=F64).view(1, 1, hd)
        exp = torch.tensor([float(v) for v in vout], dtype=F64).view(1, 1, hd)
        got = O.rope(t, torch.tensor([pos]), theta)
        assert torch.allclose(got, exp, atol=2e-9), line
        n_cases += 1
    assert n_cases >= 5


def test_p3_rope_properties():
    torch.manual_seed(0)
    q = torch.randn(1, 3, 16, dtype=F64)
    k = torch.randn(1, 3, 16, dtype=F64)
    assert torch.equal(O.rope(q, torch.tensor([0]), 1e4), q)                       # pos 0 = identity
    for p, s in [(5, 2), (130, 77), (1023, 1000)]:
        qp, ks = O.rope(q, torch.tensor([p]), 1e4), O.rope(k, torch.tensor([s]), 1e4)
        assert torch.allclose(qp.norm(dim=-1), q.norm(dim=-1))                     # rotation preserves norm
        qd = O.rope(q, torch.tensor([p - s]), 1e4)                                 # <R_p q, R_s k> = <R_{p-s} q, k>
        assert torch.allclose((qp * ks).sum(-1), (qd * k).sum(-1), atol=1e-10)
    # per-token positions: row i uses pos[i], not its row index
    t = torch.randn(3, 2, 8, dtype=F64)
    a = O.rope(t, torch.tensor([7, 3, 11]), 1e4)
    for i, p in enumerate([7, 3, 11]):
        assert torch.equal(a[i:i + 1], O.rope(t[i:i + 1], torch.tensor([p]), 1e4))


# ---------------------------------------------------------------- P4 attention special cases
def test_p4_attention_one_key_and_uniform_weights():
    torch.manual_seed(1)
    q = torch.randn(2, 8, dtype=F64)
    K = torch.randn(5, 2, 8, dtype=F64)
    V = torch.randn(5, 2, 8, dtype=F64)
    assert torch.allclose(O.attend_row(q, K[:1], V[:1]), V[0])                     # one key -> that value
    o = O.attend_row(torch.zeros(2, 8, dtype=F64), K, V)                            # q = 0 -> uniform -> mean of v
    assert torch.allclose(o, V.mean(dim=0))
    # shift invariance of softmax: adding the same vector to every key along q's direction changes nothing
    o1 = O.attend_row(q, K, V)
    o2 = O.attend_row(q, K + 3.0 * q[None] / (q * q).sum(-1, keepdim=True)[None], V)
    assert torch.allclose(o1, o2, atol=1e-12)


def test_p4_prefill_attention_equals_torch_sdpa():
    torch.manual_seed(2)
    n, H, hd = 19, 3, 16
    q, k, v = (torch.randn(n, H, hd, dtype=F64) for _ in range(3))
    ref = torch.nn.functional.scaled_dot_product_attention(
        q.permute(1, 0, 2)[None], k.permute(1, 0, 2)[None], v.permute(1, 0, 2)[None], is_causal=True)[0].permute(1, 0, 2)
    got = torch.stack([O.attend_row(q[i], k[: i + 1], v[: i + 1]) for i in range(n)])
    assert torch.allclose(got, ref, atol=1e-12)


def test_p4_zero_wq_gives_running_mean_of_v():
    cfg = SMALL
    w = I.make_weights(cfg, seed=3)
    for L in w["layers"]:
        L["wq"].zero_()
    o = O.Oracle(I.ModelCfg(**{**cfg.as_dict(), "n_layers": 1}), w, F64)
    e = I.make_embeds(cfg, 3, 0, 6)
    L = w["layers"][0]
    hid = o.step([(0, 0, 0, 6)], e)
    x = e.double()
    v = (O.rmsnorm(x, L["g_attn"].double(), cfg.rms_eps) @ L["wv"].double().T)
    run_mean = torch.cumsum(v, 0) / torch.arange(1, 7, dtype=F64)[:, None]
    x1 = x + run_mean @ L["wo"].double().T
    xn = O.rmsnorm(x1, L["g_mlp"].double(), cfg.rms_eps)
    g = xn @ L["w_gate"].double().T
    exp = x1 + ((g * torch.sigmoid(g)) * (xn @ L["w_up"].double().T)) @ L["w_down"].double().T
    assert relerr(hid, exp) < 1e-12


# ---------------------------------------------------------------- P5 identity layer (residual wiring)
def test_p5_identity_layer_and_logits_formula():
    cfg = SMALL
    w = I.make_weights(cfg, seed=4)
    for L in w["layers"]:
        L["wo"].zero_()
        L["w_down"].zero_()
    o = O.Oracle(cfg, w, F64)
    e = I.make_embeds(cfg, 4, 0, 7)
    hid = o.step([(1, 0, 0, 7)], e)
    assert torch.equal(hid, e.double())                                            # bitwise: x + 0 + 0
    K0, V0 = o.cache(0, 1)
    xn = O.rmsnorm(e.double(), w["layers"][0]["g_attn"].double(), cfg.rms_eps)
    assert torch.allclose(V0.reshape(7, -1), xn @ w["layers"][0]["wv"].double().T)  # K/V still appended
    lg = o.logits(hid, [6, 0])
    x = e.double()[[6, 0]]
    exp = (x * w["g_final"].double() / torch.sqrt((x * x).mean(1, keepdim=True) + cfg.rms_eps)) @ w["w_lm"].double().T
    assert torch.allclose(lg, exp, atol=1e-12)


# ---------------------------------------------------------------- P6 HF LlamaModel as a black box (A1, A2, A5, A16)
def test_p6_matches_transformers_llama():
    tf = pytest.importorskip("transformers")
    cfg = I.CFG_TINY
    w = I.make_weights(cfg, seed=0)
    hc = tf.LlamaConfig(hidden_size=cfg.d_model, num_hidden_layers=cfg.n_layers, num_attention_heads=cfg.n_heads,
                        num_key_value_heads=cfg.n_heads, intermediate_size=cfg.ffn, rms_norm_eps=cfg.rms_eps,
                        rope_theta=cfg.rope_theta, vocab_size=cfg.vocab, max_position_embeddings=256,
                        attention_bias=False, mlp_bias=False, hidden_act="silu")
    hc._attn_implementation = "eager"
    model = tf.LlamaModel(hc).to(torch.float64).eval()
    sd = {}
    names = {"wq": "self_attn.q_proj", "wk": "self_attn.k_proj", "wv": "self_attn.v_proj", "wo": "self_attn.o_proj",
             "w_gate": "mlp.gate_proj", "w_up": "mlp.up_proj", "w_down": "mlp.down_proj",
             "g_attn": "input_layernorm", "g_mlp": "post_attention_layernorm"}
    for l, L in enumerate(w["layers"]):
        for k, hf in names.items():
            sd[f"layers.{l}.{hf}.weight"] = L[k].double()
    sd["norm.weight"] = w["g_final"].double()
    sd["embed_tokens.weight"] = model.state_dict()["embed_tokens.weight"]
    missing = model.load_state_dict(sd, strict=False)
    assert not [m for m in missing.missing_keys if "rotary" not in m]
    e = I.make_embeds(cfg, 0, 0, 21)
    with torch.no_grad():
        out = model(inputs_embeds=e.double()[None], use_cache=True)
        ref_prefill = out.last_hidden_state[0]                                   # final-normed hidden
        e2 = I.make_embeds(cfg, 0, 1, 1)
        out2 = model(inputs_embeds=e2.double()[None], past_key_values=out.past_key_values, use_cache=True,
                     position_ids=torch.tensor([[21]]))
        ref_dec = out2.last_hidden_state[0]
    o = O.Oracle(cfg, w, F64)
    hid = o.step([(0, 0, 0, 21)], e)
    hid2 = o.step([(0, 1, 21, 1)], e2)
    g = w["g_final"].double()
    # HF builds its cos/sin tables from a float32 inv_freq buffer, so agreement is to fp32 rounding (~1e-7), not
    # fp64; a wrong pairing, sign, residual wiring or weight layout gives O(1) error.
    assert relerr(O.rmsnorm(hid, g, cfg.rms_eps), ref_prefill) < 2e-6
    assert relerr(O.rmsnorm(hid2, g, cfg.rms_eps), ref_dec) < 2e-6


# ---------------------------------------------------------------- P7 oracle invariants
def test_p7_prefill_then_decode_equals_prefill_of_concatenation_and_chunking():
    cfg = I.CFG_TINY
    w = I.make_weights(cfg, seed=0)
    e = I.make_embeds(cfg, 0, 7, 31)
    one = O.Oracle(cfg, w, F64).step([(0, 0, 0, 31)], e)
    o = O.Oracle(cfg, w, F64)
    a = o.step([(2, 0, 0, 30)], e[:30])
    b = o.step([(2, 1, 30, 1)], e[30:])
    assert relerr(torch.cat([a, b]), one) < 1e-12
    o = O.Oracle(cfg, w, F64)                                                     # chunked prefill 11 + 13 + 7
    parts = [o.step([(1, 0, 0, 11)], e[:11]), o.step([(1, 0, 11, 13)], e[11:24]), o.step([(1, 0, 24, 7)], e[24:])]
    assert relerr(torch.cat(parts), one) < 1e-12


def test_p7_requests_are_independent_and_order_is_immaterial():
    cfg = I.CFG_TINY
    w = I.make_weights(cfg, seed=0)
    eA, eB = I.make_embeds(cfg, 0, 1, 9), I.make_embeds(cfg, 0, 2, 5)
    o1 = O.Oracle(cfg, w, F64)
    h1 = o1.step([(0, 0, 0, 9), (1, 0, 0, 5)], torch.cat([eA, eB]))
    o2 = O.Oracle(cfg, w, F64)
    h2 = o2.step([(1, 0, 0, 5), (0, 0, 0, 9)], torch.cat([eB, eA * 3]))           # A perturbed, order swapped
    assert torch.equal(h1[9:], h2[:5])                                            # B's rows unchanged, bitwise


# ---------------------------------------------------------------- P10/P11 library steps and SiLU values
def test_p10_matmul_against_triple_loop():
    torch.manual_seed(3)
    a, b = torch.randn(7, 13, dtype=F64), torch.randn(29, 13, dtype=F64)
    ref = torch.zeros(7, 29, dtype=F64)
    for i in range(7):
        for j in range(29):
            s = 0.0
            for k in range(13):
                s += float(a[i, k]) * float(b[j, k])
            ref[i, j] = s
    assert torch.allclose(a @ b.T, ref, atol=1e-12)


def test_p11_silu_values():
    z = torch.tensor([0.0, 1.0, -1.0, 100.0, -100.0], dtype=F64)
    s = O.silu(z)
    assert s[0] == 0.0
    assert abs(float(s[1]) - 0.7310585786) < 1e-9
    assert abs(float(s[2]) + 0.2689414214) < 1e-9
    assert float(s[3]) == 100.0 and abs(float(s[4])) < 1e-40 and torch.isfinite(s).all()


def test_argmax_rows_ties_nans_and_library_routine():
    """oracle.argmax_rows against what fixes it: hand-made rows (ties -> lowest index, NaNs skipped, all -inf / all
    NaN -> 0) and, on random rows without ties, numpy's argmax."""
    import numpy as np
    nan, inf = float("nan"), float("inf")
    rows = torch.tensor([[1.0, 3.0, 3.0, 2.0], [nan, -1.0, nan, -1.0], [-inf, -inf, -inf, -inf], [nan, nan, nan, nan],
                         [0.0, -0.0, 0.0, -0.0], [5.0, 1.0, inf, inf]])
    assert O.argmax_rows(rows) == [1, 1, 0, 0, 0, 2]
    g = torch.Generator().manual_seed(3)
    r = torch.randn(9, 1000, generator=g)
    assert O.argmax_rows(r) == [int(i) for i in np.argmax(r.numpy(), axis=1)]


def test_embed_rows_is_a_row_gather():
    g = torch.Generator().manual_seed(4)
    table = torch.randn(50, 16, generator=g).to(torch.bfloat16)
    toks = [3, 49, 0, 3, 50, -1]
    out = O.embed_rows(table, toks)
    assert torch.equal(out[:4], table[torch.tensor(toks[:4])]) and not out[4:].any()


# ---------------------------------------------------------------- f1: Algorithm 1's token loop
def _frame_inputs(cfg, n_frames, L_P):
    g = torch.Generator().manual_seed(31)
    table = (torch.randn(cfg.vocab, cfg.d_model, generator=g)).to(torch.bfloat16)
    return table, [I.make_embeds(cfg, 31, f, L_P) for f in range(n_frames)]


def test_greedy_frame_equals_bruteforce_recomputation():
    """greedy_frame pinned by brute force: at every stage s the logits equal LMHead(Norm(.)) of the last row of a
    cache-free full-sequence forward over [prefill rows ; Embed(a_0) .. Embed(a_{s-1})] and the token is numpy's argmax."""
    import numpy as np
    cfg, L_P, K = SMALL, 11, 5
    w = I.make_weights(cfg, seed=7)
    table, frames = _frame_inputs(cfg, 1, L_P)
    o = O.Oracle(cfg, w, F64)
    toks, lg = O.greedy_frame(o, 2, frames[0], table, K)
    seq = frames[0].to(F64)
    for s in range(K):
        hid = O.brute_forward(cfg, w, seq)
        hn = O.rmsnorm(hid[-1:], w["g_final"].to(F64), cfg.rms_eps)
        ref = (hn @ w["w_lm"].to(F64).T)[0]
        assert relerr(lg[s], ref) < 1e-9
        assert toks[s] == int(np.argmax(ref.to(torch.float32).numpy()))
        seq = torch.cat([seq, table[toks[s]][None].to(F64)])
    # teacher forcing feeds the given tokens, and reports the oracle's own argmax at each stage
    forced = [(t + 1) % cfg.vocab for t in toks]
    toks_f, lg_f = O.greedy_frame(o, 2, frames[0], table, K, forced=forced)
    assert toks_f[0] == toks[0] and relerr(lg_f[0], lg[0]) < 1e-12
    seq = torch.cat([frames[0].to(F64), table[forced[0]][None].to(F64)])
    hn = O.rmsnorm(O.brute_forward(cfg, w, seq)[-1:], w["g_final"].to(F64), cfg.rms_eps)
    assert relerr(lg_f[1], (hn @ w["w_lm"].to(F64).T)[0]) < 1e-9


def test_pipelined_loop_equals_sequential_frames():
    """The paper's claim the loop rests on ("functionally lossless"): running Alg. 1 as the K-stage pipeline
    (steady_schedule, tokens of step t feeding the decode rows of step t+1, regions recycled) gives every frame the
    tokens and logits of that frame run alone by greedy_frame."""
    cfg, L_P, K, R, n_frames = SMALL, 9, 4, 5, 9
    w = I.make_weights(cfg, seed=8)
    table, frames = _frame_inputs(cfg, n_frames, L_P)
    alone = O.Oracle(cfg, w, F64)
    want = [O.greedy_frame(alone, 0, frames[f], table, K) for f in range(n_frames)]
    o = O.Oracle(cfg, w, F64)
    got_tok = [[None] * K for _ in range(n_frames)]
    prev = []                                             # tokens of the previous step, by stage
    for t in range(n_frames + K - 1):
        segs = [s for s in I.steady_schedule(t, L_P, K, R) if (t - (s[2] - L_P + 1 if s[1] else 0)) < n_frames]
        dec = [s for s in segs if s[1] == 1]
        pre = [s for s in segs if s[1] == 0]
        rows, stages = [], []
        if pre:
            o.reset(pre[0][0])
            rows.append(frames[t]); stages.append(0)
        for s in dec:
            st = s[2] - L_P + 1
            rows.append(O.embed_rows(table, [prev[st - 1]])); stages.append(st)
        hid = o.step(segs, torch.cat(rows))
        lg = o.logits(hid, I.prediction_rows(segs))
        toks = O.argmax_rows(lg.to(torch.float32))
        cur = [None] * K
        for i, st in enumerate(stages):
            f = t - st
            got_tok[f][st] = toks[i]
            cur[st] = toks[i]
            assert relerr(lg[i], want[f][1][st]) < 1e-9, (t, st)
        prev = cur
    assert got_tok == [w_[0] for w_ in want]


# ---------------------------------------------------------------- f3: sliding window inside a request
def test_window_oracle_against_banded_bruteforce_and_special_cases():
    """Oracle(window=W) pinned by (1) the cache-free brute force with an explicit banded mask, fed in chunks that the
    ring rule allows (chunk <= C - W + 1 is a ring matter; the oracle takes any chunking), (2) W >= n == no window,
    (3) W = 1: every row sees only itself, so attention returns its own v and the layer has a closed form."""
    cfg, n = SMALL, 37
    w = I.make_weights(cfg, seed=9)
    e = I.make_embeds(cfg, 9, 0, n)
    for W in (1, 5, 16):
        ref = O.brute_forward(cfg, w, e, window=W)
        o = O.Oracle(cfg, w, F64, window=W)
        got, p = [], 0
        for chunk in (7, 1, 1, 12, 1, 15):
            got.append(o.step([(0, 0 if chunk > 1 else 1, p, chunk)], e[p:p + chunk]))
            p += chunk
        assert p == n and relerr(torch.cat(got), ref) < 1e-9, W
    full = O.Oracle(cfg, w, F64).step([(0, 0, 0, n)], e)
    assert relerr(O.Oracle(cfg, w, F64, window=n).step([(0, 0, 0, n)], e), full) < 1e-12
    assert relerr(O.Oracle(cfg, w, F64, window=n + 50).step([(0, 0, 0, n)], e), full) < 1e-12
    assert relerr(O.brute_forward(cfg, w, e, window=n), O.brute_forward(cfg, w, e)) < 1e-12
    # W = 1 closed form, one layer: o = v (softmax over one key), position-independent (RoPE cancels in q.k, v unrotated)
    one = I.ModelCfg(d_model=64, n_layers=1, n_heads=4, head_dim=16, ffn=80, vocab=40)
    w1 = I.make_weights(one, seed=10)
    L = {k: v.to(F64) for k, v in w1["layers"][0].items()}
    x = I.make_embeds(one, 10, 0, 6).to(F64)
    xn = O.rmsnorm(x, L["g_attn"], one.rms_eps)
    h = x + (xn @ L["wv"].T) @ L["wo"].T
    hn = O.rmsnorm(h, L["g_mlp"], one.rms_eps)
    want = h + (O.silu(hn @ L["w_gate"].T) * (hn @ L["w_up"].T)) @ L["w_down"].T
    assert relerr(O.Oracle(one, w1, F64, window=1).step([(3, 0, 0, 6)], x.to(torch.bfloat16)), want) < 1e-12


def test_window_index_model_rules():
    """f3 ring rule: with a window W a request may outgrow its region; a segment that wraps past C must satisfy
    len <= C - W + 1 (its first row's window must survive its last row's append); brute force over a small ring that
    the slot of every position a row may attend still holds that position after the step's appends."""
    R, C = 2, 8
    for W in (1, 3, 8):
        for start in range(0, 20):
            for n in range(1, 9):
                base, length = [5, 0], [start, 0]
                try:
                    _, pos, slot, new_len = O.ring_index_model(R, C, base, length, [(0, 0, start, n)], window=W, max_pos=24)
                except ValueError as ex:
                    assert str(ex) == "AF_ERR_CAPACITY"
                    assert start + n > 24 or (start + n > C and n > C - W + 1)
                    continue
                # contents after the appends: slot -> newest position written there
                held = {}
                for p in range(0, start + n):
                    held[(base[0] + p) % C] = p
                for p in pos:
                    for j in range(max(0, p - W + 1), p + 1):
                        assert held[(base[0] + j) % C] == j, (W, start, n, p, j)
                assert new_len[0] == start + n
    # without a window the v1 rule stands
    with pytest.raises(ValueError):
        O.ring_index_model(R, C, [0, 0], [7, 0], [(0, 1, 7, 1), (1, 0, 0, 9)])
