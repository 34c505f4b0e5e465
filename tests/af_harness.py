"""Test harness: drives the CUDA path (through the C ABI binding) and the oracle with identical seeded inputs."""
import os

import torch

from oracle import af_oracle as O
from paper_2512_20276_b200 import inputs as I

TOL = 2e-2          # BASELINE.json north_star: max|err| <= 2e-2 * max|ref| per compared tensor

# The oracle's tiny per-row ops collapse when torch's OpenMP pool oversubscribes the container's cores.
torch.set_num_threads(max(1, (os.cpu_count() or 4) - 2))


def relmax(got: torch.Tensor, ref: torch.Tensor) -> float:
    ref = ref.double().cpu()
    return float((got.double().cpu() - ref).abs().max() / ref.abs().max())


class Pair:
    """One CUDA ring + one oracle fed the same steps; checks bookkeeping bit-exactly and tensors to TOL."""

    def __init__(self, cfg, host_weights, R, C, max_rows, bases=None, oracle_dtype=torch.float64, dev_weights=None,
                 window=0, max_pos=0):
        from paper_2512_20276_b200 import binding
        self.binding = binding
        self.cfg, self.R, self.C = cfg, R, C
        self.W = dev_weights if dev_weights is not None else binding.Weights(cfg, host_weights)
        self.ring = binding.Ring(cfg, R, C, max_rows=max_rows)
        self.window, self.max_pos = window, max_pos
        if window:
            self.ring.set_window(window, max_pos)                      # f3: sliding window inside a request
        self.orc = O.Oracle(cfg, host_weights, oracle_dtype, window=window or None)
        self.base = [0] * R
        self.len = [0] * R
        if bases is not None:
            for r, b in enumerate(bases):
                self.reset(r, b)

    def reset(self, req, new_base=-1):
        self.ring.reset_slot(req, new_base)
        self.orc.reset(req)
        self.base[req], self.len[req] = O.ring_reset_model(self.C, self.base[req], self.len[req], new_base)
        assert self.ring.get_state(req) == (self.base[req], self.len[req])

    def step(self, segs, embeds, check=True, oracle=True):
        """Returns (gpu_hidden, oracle_hidden or None)."""
        hid = self.ring.packed_forward(self.W, embeds.cuda(), segs)
        mr, mp, ms, new_len = O.ring_index_model(self.R, self.C, self.base, self.len, segs, self.window, self.max_pos)
        rr, rp, rs = self.ring.row_map(len(mr))
        assert (rr, rp, rs) == (mr, mp, ms), "device row map differs from the index model (must be bit-exact)"
        self.len = new_len
        for r in range(self.R):
            assert self.ring.get_state(r) == (self.base[r], self.len[r])
        ref = None
        if oracle:
            ref = self.orc.step(segs, embeds)
            if check:
                err = relmax(hid, ref)
                assert err <= TOL, f"hidden max|err|/max|ref| = {err:.3e}"
        return hid, ref

    def check_ring(self, reqs, layers=None):
        """Ring K/V of every live slot, read in logical order (base + j) mod C, against the oracle's linear cache."""
        kv = self.ring.kv_view()
        worst = 0.0
        for l in (layers if layers is not None else range(self.cfg.n_layers)):
            for r in reqs:
                n = self.len[r]
                if n == 0:
                    continue
                lo = max(0, n - self.C)                                # older positions were overwritten (f3)
                slots = torch.tensor([(self.base[r] + j) % self.C for j in range(lo, n)], device=kv.device)
                Kc, Vc = self.orc.cache(l, r)
                Kc, Vc = Kc[lo:], Vc[lo:]
                k_gpu = kv[l, 0, r].index_select(1, slots).permute(1, 0, 2)     # [n, H, hd]
                v_gpu = kv[l, 1, r].index_select(1, slots).permute(1, 0, 2)
                worst = max(worst, relmax(k_gpu, Kc), relmax(v_gpu, Vc))
        assert worst <= TOL, f"ring K/V max|err|/max|ref| = {worst:.3e}"
        return worst

    def check_logits(self, hid, ref, rows):
        lg = self.ring.logits_rows(self.W, hid, rows)
        ref_lg = self.orc.logits(ref, rows)
        err = relmax(lg, ref_lg)
        assert err <= TOL, f"logits max|err|/max|ref| = {err:.3e}"
        return lg, ref_lg
