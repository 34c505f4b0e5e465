"""ORACLE — test infrastructure, not product code.

Plain, slow CPU statement of what the Cross-Request State Packed Forward (ActionFlow, arxiv 2512.20276,
Algorithm 2) must compute.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this file; it imports nothing from the CUDA package and shares no code with it.

The method is an exact re-scheduling ("functionally lossless" against sequential inference),
so the oracle is the plain definition: EVERY MICRO-REQUEST IS RUN ALONE AND UNPACKED through a standard
Llama-style decoder with its own contiguous, linearly indexed KV cache (the paper's "Baseline" schedule).
No ring, no packing, no segment mask.  Library primitives used as steps: torch CPU matmul / exp / softmax-free
explicit formulas.  dtype: float64 by default (tiny configs); float32 for 7B shapes as BASELINE.json's
north_star fixes ("a plain fp32 CPU implementation"), with RMSNorm's sum of squares and the softmax in the
working dtype.  Inputs are the bf16-rounded weights/embeddings widened to the working dtype; no intermediate
is rounded to bf16 (that rounding is the CUDA path's error budget).

Pins (tests/test_oracle_pins.py): brute-force full-sequence recomputation (brute_forward, below, which has no
cache and an explicit mask), RMSNorm / RoPE / SiLU closed forms and worked values, attention special cases
(one key, zero Wq -> running mean, torch SDPA), identity layer, HF transformers LlamaModel as a black box,
prefill-then-decode == prefill of the concatenation, chunked prefill, request independence, ring-index brute
force; greedy_frame (Alg. 1's token loop) by brute-force recomputation of every stage and by "the K-stage pipeline
gives every frame the tokens of that frame run alone".  Parity unpinned: the paper prints no numeric worked example of any forward quantity; eps, theta and
the rotate-half RoPE pairing come from BASELINE.json configs[0] and the HF-Llama convention (A2, A5).
"""
from __future__ import annotations

import math

import torch


def _w(t: torch.Tensor, dtype) -> torch.Tensor:
    return t.to(dtype)


# ------------------------------------------------------------------------------------------------- steps
def rmsnorm(x: torch.Tensor, g: torch.Tensor, eps: float) -> torch.Tensor:
    """O1/O7 (Alg. 2 l.1; reading A2): x * g / sqrt(mean(x^2) + eps), no mean subtraction, no bias."""
    ms = (x * x).sum(dim=-1, keepdim=True) / x.shape[-1]
    return x * g / torch.sqrt(ms + eps)


def rope(t: torch.Tensor, pos: torch.Tensor, theta: float) -> torch.Tensor:
    """O3 (Alg. 2 l.3; reading A5): rotate-half RoPE.  t: [n, H, hd], pos: [n] integer positions
    "within the original request".  f_c = theta^(-2c/hd); t'[c] = t[c] cos - t[c+hd/2] sin;
    t'[c+hd/2] = t[c+hd/2] cos + t[c] sin.  Angles are formed in float64 and cast to t's dtype."""
    n, H, hd = t.shape
    half = hd // 2
    c = torch.arange(half, dtype=torch.float64)
    f = torch.pow(torch.tensor(float(theta), dtype=torch.float64), -2.0 * c / hd)
    a = pos.to(torch.float64)[:, None] * f[None, :]              # [n, half]
    cos = torch.cos(a).to(t.dtype)[:, None, :]
    sin = torch.sin(a).to(t.dtype)[:, None, :]
    lo, hi = t[..., :half], t[..., half:]
    return torch.cat([lo * cos - hi * sin, hi * cos + lo * sin], dim=-1)


def silu(z: torch.Tensor) -> torch.Tensor:
    """silu(z) = z / (1 + exp(-z))  (O8)."""
    return z / (1.0 + torch.exp(-z))


def attend_row(q: torch.Tensor, Kc: torch.Tensor, Vc: torch.Tensor) -> torch.Tensor:
    """O5 (Alg. 2 l.4; reading A9) for ONE query row against ITS OWN request's cache prefix.
    q: [H, hd]; Kc, Vc: [ctx, H, hd] = cache positions 0..p (inclusive of the row's own position).
    s_j = q.k_j / sqrt(hd); w = exp(s - max s); o = sum_j w_j v_j / sum_j w_j."""
    hd = q.shape[-1]
    s = torch.einsum("hd,jhd->hj", q, Kc) / math.sqrt(hd)        # [H, ctx]
    m = s.max(dim=-1, keepdim=True).values
    w = torch.exp(s - m)
    o = torch.einsum("hj,jhd->hd", w, Vc) / w.sum(dim=-1)[:, None]
    return o


# ------------------------------------------------------------------------------------------------ oracle
class Oracle:
    """Runs each micro-request separately, unpacked, with a private contiguous KV cache per (layer, request)."""

    def __init__(self, cfg, weights: dict, dtype=torch.float64, cache_widened: bool = True, window=None):
        self.cfg = cfg
        # f3 ("updates the ring buffer's sliding window, discarding stale tokens"; A8b): with a window W
        # the row at position p sees positions max(0, p - W + 1)..p of its own request, nothing older.  The oracle's
        # cache stays linear and unbounded: "wrap == linear window".  None = the whole prefix (v1 semantics).
        self.window = window
        self.w = weights            # bf16 (or float) CPU tensors, widened to the working dtype on use
        self.dtype = dtype
        self._wide = {} if cache_widened else None   # id(tensor) -> widened copy (same values, kept between calls)
        self.K = {}                 # (layer, req) -> [pos, H, hd]
        self.V = {}
        self.len = {}               # req -> tokens cached

    def _widen(self, t: torch.Tensor, dtype) -> torch.Tensor:
        if self._wide is None or t.dtype == dtype:
            return t.to(dtype)
        k = id(t)
        if k not in self._wide:
            self._wide[k] = t.to(dtype)
        return self._wide[k]

    # -- request lifecycle -------------------------------------------------------------------------------
    def reset(self, req: int):
        """A finished request is evicted and its id reused: drop its private cache."""
        for l in range(self.cfg.n_layers):
            self.K.pop((l, req), None)
            self.V.pop((l, req), None)
        self.len[req] = 0

    def ctx_len(self, req: int) -> int:
        return self.len.get(req, 0)

    # -- one segment = one micro-request advanced alone --------------------------------------------------
    def run_segment(self, req: int, start_pos: int, x_in: torch.Tensor) -> torch.Tensor:
        cfg, dt = self.cfg, self.dtype
        H, hd = cfg.n_heads, cfg.head_dim
        n = x_in.shape[0]
        _w = self._widen
        assert start_pos == self.ctx_len(req), "appends must be contiguous (O0)"
        x = x_in.to(dt)                                                    # O0
        pos = torch.arange(start_pos, start_pos + n)
        for l in range(cfg.n_layers):
            L = self.w["layers"][l]
            xn = rmsnorm(x, _w(L["g_attn"], dt), cfg.rms_eps)              # O1
            q = (xn @ _w(L["wq"], dt).T).view(n, H, hd)                    # O2
            k = (xn @ _w(L["wk"], dt).T).view(n, H, hd)
            v = (xn @ _w(L["wv"], dt).T).view(n, H, hd)
            q = rope(q, pos, cfg.rope_theta)                               # O3
            k = rope(k, pos, cfg.rope_theta)
            if start_pos == 0:                                             # O4: linear index = position
                Kc, Vc = k, v
            else:
                Kc = torch.cat([self.K[(l, req)], k], dim=0)
                Vc = torch.cat([self.V[(l, req)], v], dim=0)
            self.K[(l, req)], self.V[(l, req)] = Kc, Vc
            o = torch.empty(n, H, hd, dtype=dt)
            for i in range(n):                                             # O5: row i sees positions 0..p_i
                p = start_pos + i
                lo = 0 if self.window is None else max(0, p - self.window + 1)
                o[i] = attend_row(q[i], Kc[lo: p + 1], Vc[lo: p + 1])
            x = x + o.reshape(n, H * hd) @ _w(L["wo"], dt).T               # O6 (reading A1)
            xn2 = rmsnorm(x, _w(L["g_mlp"], dt), cfg.rms_eps)              # O7
            g = xn2 @ _w(L["w_gate"], dt).T
            u = xn2 @ _w(L["w_up"], dt).T
            x = x + (silu(g) * u) @ _w(L["w_down"], dt).T                  # O8
        self.len[req] = start_pos + n
        return x

    def step(self, segs, embeds: torch.Tensor) -> torch.Tensor:
        """All segments of one computation batch, one at a time (requests are disjoint, order immaterial).
        segs: [(req_id, phase, start_pos, len)], embeds: [T, D] rows in segment order. Returns hidden [T, D]."""
        T = sum(s[3] for s in segs)
        assert embeds.shape[0] == T
        out = torch.empty(T, self.cfg.d_model, dtype=self.dtype)
        r0 = 0
        for (req, _phase, start, n) in segs:
            out[r0:r0 + n] = self.run_segment(req, start, embeds[r0:r0 + n])
            r0 += n
        return out

    def logits(self, hidden: torch.Tensor, rows) -> torch.Tensor:
        """O9 (Alg. 1 l.5/l.8): RMSNorm(hidden[rows]; g_final) W_lm^T."""
        dt = self.dtype
        _w = self._widen
        h = hidden[list(rows)].to(dt)
        hn = rmsnorm(h, _w(self.w["g_final"], dt), self.cfg.rms_eps)
        return hn @ _w(self.w["w_lm"], dt).T

    def cache(self, layer: int, req: int):
        """(K, V) of request req at layer, each [len, H, hd], index = logical position."""
        return self.K[(layer, req)], self.V[(layer, req)]


# ------------------------------------------------------------------------------------- brute-force mode
def brute_forward(cfg, weights: dict, embeds: torch.Tensor, window=None) -> torch.Tensor:
    """Pin P1: ONE request of n tokens recomputed with NO cache — full forward over rows 0..n-1 with an explicit
    n x n causal mask, float64 throughout, written independently of Oracle.run_segment (masked dense softmax
    instead of per-row prefixes; explicit per-pair rotation instead of the vectorised rope())."""
    dt = torch.float64
    n, D = embeds.shape
    H, hd = cfg.n_heads, cfg.head_dim
    half = hd // 2
    x = embeds.to(dt)
    mask = torch.zeros(n, n, dtype=torch.bool)
    for i in range(n):
        for j in range(n):
            mask[i, j] = j <= i and (window is None or i - j < window)      # banded when a window is given (f3)
    ang = torch.zeros(n, half, dtype=dt)
    for p in range(n):
        for c in range(half):
            ang[p, c] = p * (cfg.rope_theta ** (-2.0 * c / hd))

    def rot(t):                                    # t: [n, H, hd]
        out = torch.empty_like(t)
        for c in range(half):
            cs, sn = torch.cos(ang[:, c])[:, None], torch.sin(ang[:, c])[:, None]
            out[:, :, c] = t[:, :, c] * cs - t[:, :, c + half] * sn
            out[:, :, c + half] = t[:, :, c + half] * cs + t[:, :, c] * sn
        return out

    for l in range(cfg.n_layers):
        L = {k: v.to(dt) for k, v in weights["layers"][l].items()}
        xn = x * L["g_attn"] / torch.sqrt((x ** 2).mean(dim=1, keepdim=True) + cfg.rms_eps)
        q = rot((xn @ L["wq"].T).view(n, H, hd))
        k = rot((xn @ L["wk"].T).view(n, H, hd))
        v = (xn @ L["wv"].T).view(n, H, hd)
        att = torch.empty(n, H, hd, dtype=dt)
        for h in range(H):
            s = (q[:, h, :] @ k[:, h, :].T) / math.sqrt(hd)
            s = s.masked_fill(~mask, float("-inf"))
            p = torch.softmax(s, dim=1)
            att[:, h, :] = p @ v[:, h, :]
        x = x + att.reshape(n, D) @ L["wo"].T
        xn = x * L["g_mlp"] / torch.sqrt((x ** 2).mean(dim=1, keepdim=True) + cfg.rms_eps)
        gate = xn @ L["w_gate"].T
        x = x + ((gate * torch.sigmoid(gate)) * (xn @ L["w_up"].T)) @ L["w_down"].T
    return x


# ------------------------------------------------------------------------------------- ring index model
def ring_index_model(R: int, C: int, base, length, segs, window=0, max_pos=0):
    """Pure-integer model of step a0 / reading A6 (BASELINE.json north_star: "slot (base_r + pos) mod capacity
    of its request's region").  Returns (row_req, row_pos, row_slot, new_length) or raises ValueError with the
    AF_ERR_* name the library must return.  row_slot = req*C + ((base[req] + pos) mod C)."""
    seen = set()
    for (req, phase, start, n) in segs:
        if not (0 <= req < R) or req in seen or n < 1 or (phase == 1 and n != 1) or phase not in (0, 1):
            raise ValueError("AF_ERR_SEGMENT")
        seen.add(req)
    for (req, phase, start, n) in segs:
        if start != length[req]:
            raise ValueError("AF_ERR_POSITION")
    for (req, phase, start, n) in segs:
        if window <= 0:
            if start + n > C:
                raise ValueError("AF_ERR_CAPACITY")
        else:
            # f3: a request may outgrow its region; slot (base + pos) mod C then overwrites position pos - C.  Every row
            # of the step is appended before any row attends, so the first row's window (start - W + 1 ..) must survive
            # the last row's append (which evicts start + n - 1 - C): n <= C - W + 1.  Positions stay below max_pos.
            if start + n > (max_pos if max_pos > 0 else C) or (start + n > C and n > C - window + 1):
                raise ValueError("AF_ERR_CAPACITY")
    row_req, row_pos, row_slot = [], [], []
    new_len = list(length)
    for (req, phase, start, n) in segs:
        for i in range(n):
            pos = start + i
            row_req.append(req)
            row_pos.append(pos)
            row_slot.append(req * C + ((base[req] + pos) % C))
        new_len[req] = start + n
    return row_req, row_pos, row_slot, new_len


def ring_reset_model(C: int, base: int, length: int, new_base: int):
    """af_ring_reset_slot bookkeeping: returns (base, len) after recycling a region."""
    if new_base >= 0:
        return new_base % C, 0
    return (base + length) % C, 0


def argmax_rows(logits) -> list:
    """Alg. 1 l.5 / l.8 "ArgMax(LMHead(Norm(H[s])))" as the plain definition, one scalar loop per row:
    the LOWEST index whose value is the row maximum; NaN entries are never selected (a row of only NaNs gives 0).
    The decision is taken on the logits exactly as given (fp32), which is the precision the library decides in."""
    out = []
    for row in logits.tolist():
        best, best_i = float("-inf"), -1
        for i, v in enumerate(row):
            if v > best or (v == best and best_i < 0):
                best, best_i = v, i
        out.append(max(best_i, 0))
    return out


def embed_rows(table: torch.Tensor, tokens) -> torch.Tensor:
    """The token half of Alg. 1 l.2 "Embed(.., GetLastTokenEach(A_sequences))": row i = table[tokens[i]]
    (a token outside the table gives a row of zeros, as the library documents)."""
    out = torch.zeros(len(tokens), table.shape[1], dtype=table.dtype)
    for i, t in enumerate(tokens):
        if 0 <= int(t) < table.shape[0]:
            out[i] = table[int(t)]
    return out


def greedy_frame(oracle: "Oracle", req: int, prefill_embeds: torch.Tensor, table: torch.Tensor, K: int, forced=None):
    """Algorithm 1 for ONE frame run alone - the paper's sequential "Baseline" schedule, which the
    pipelined loop must reproduce ("functionally lossless"): prefill the frame's L_P rows,
    a_0 = ArgMax(LMHead(Norm(H[last]))) (l.5); then for s = 1..K-1 decode Embed(a_{s-1}) (l.2) at 0-indexed position
    L_P + s - 1 (A4) and take a_s the same way (l.8).  `forced`: optional K tokens fed back INSTEAD of the
    oracle's own argmax (teacher forcing, used when the caller compares logits along another implementation's token
    path).  Returns (tokens [K] the oracle's own argmax at every stage, logits [K, V])."""
    oracle.reset(req)
    L_P = prefill_embeds.shape[0]
    hid = oracle.step([(req, 0, 0, L_P)], prefill_embeds)
    lg = [oracle.logits(hid, [L_P - 1])[0]]
    toks = [argmax_rows(lg[0][None].to(torch.float32))[0]]
    for s in range(1, K):
        fed = toks[s - 1] if forced is None else int(forced[s - 1])
        x = embed_rows(table, [fed])
        hid = oracle.step([(req, 1, L_P + s - 1, 1)], x)
        lg.append(oracle.logits(hid, [0])[0])
        toks.append(argmax_rows(lg[s][None].to(torch.float32))[0])
    return toks, torch.stack(lg)
