"""Pins P8/P9: the pure-integer ring index model and the steady-state schedule values the paper prints. CPU only."""
import pytest
from hypothesis import given, settings, strategies as st

from oracle import af_oracle as O
from paper_2512_20276_b200 import inputs as I


# ------------------------------------------------------------------ P8: brute force over small rings
@pytest.mark.parametrize("C", [1, 2, 3, 8, 128])
def test_p8_slots_distinct_and_wrap_equals_linear(C):
    R = 3
    for base in range(C):
        for n in range(1, C + 1):
            segs = [(1, 0, 0, n)]
            req, pos, slot, new_len = O.ring_index_model(R, C, [0, base, 0], [0, 0, 0], segs)
            assert pos == list(range(n)) and req == [1] * n and new_len == [0, n, 0]
            assert len(set(slot)) == n                                  # no live token overwritten
            assert all(C <= s < 2 * C for s in slot)                    # stays inside region 1
            # first wrap happens exactly at pos = C - base
            wraps = [p for p in range(1, n) if slot[p] < slot[p - 1]]
            assert wraps == ([C - base] if 0 < C - base < n else [])
            # reading (base + j) mod C for j < len returns the linear sequence: a physical array indexed by slot
            phys = {}
            for p, s in zip(pos, slot):
                phys[s] = p
            assert [phys[1 * C + (base + j) % C] for j in range(n)] == list(range(n))


def test_p8_error_classes():
    R, C = 4, 8
    base, ln = [0] * R, [0, 3, 8, 0]
    for segs, err in [
        ([(4, 0, 0, 1)], "AF_ERR_SEGMENT"), ([(-1, 0, 0, 1)], "AF_ERR_SEGMENT"),
        ([(0, 0, 0, 1), (0, 1, 1, 1)], "AF_ERR_SEGMENT"), ([(0, 0, 0, 0)], "AF_ERR_SEGMENT"),
        ([(1, 1, 3, 2)], "AF_ERR_SEGMENT"), ([(1, 0, 2, 1)], "AF_ERR_POSITION"),
        ([(1, 0, 4, 1)], "AF_ERR_POSITION"), ([(1, 0, 3, 6)], "AF_ERR_CAPACITY"), ([(2, 1, 8, 1)], "AF_ERR_CAPACITY"),
    ]:
        with pytest.raises(ValueError, match=err):
            O.ring_index_model(R, C, base, ln, segs)
    assert O.ring_index_model(R, C, base, ln, []) == ([], [], [], ln)   # empty step is a legal no-op
    assert O.ring_index_model(R, C, base, ln, [(1, 0, 3, 5)])[3] == [0, 8, 8, 0]   # exactly full is legal


def test_p8_cfg1_wrap_case_from_baseline_config():
    # BASELINE.json configs[0]: C=128; B decodes at pos 70, C at pos 127 ("exercises wrap on next append").
    R, C = 4, 128
    base = [0, 100, 1, 77]
    req, pos, slot, nl = O.ring_index_model(R, C, base, [0, 70, 127, 0], [(0, 0, 0, 64), (1, 1, 70, 1), (2, 1, 127, 1)])
    assert slot[64] == 1 * C + (100 + 70) % 128 == 128 + 42
    assert slot[65] == 2 * C + (1 + 127) % 128 == 256 + 0             # lands in slot 0 of region 2
    assert nl == [64, 71, 128, 0]
    with pytest.raises(ValueError, match="AF_ERR_CAPACITY"):
        O.ring_index_model(R, C, base, nl, [(2, 1, 128, 1)])
    assert O.ring_reset_model(C, 1, 128, -1) == (1, 0)               # (1 + 128) mod 128
    assert O.ring_reset_model(C, 100, 71, -1) == (43, 0)
    assert O.ring_reset_model(C, 100, 71, 300) == (300 % 128, 0)


@settings(max_examples=200, deadline=None)
@given(st.data())
def test_p8_random_tables_never_alias_live_tokens(data):
    R = data.draw(st.integers(1, 6))
    C = data.draw(st.integers(1, 40))
    base = [data.draw(st.integers(0, C - 1)) for _ in range(R)]
    ln = [0] * R
    owner = {}                                                          # global slot -> (req, pos) of live tokens
    for _ in range(data.draw(st.integers(1, 6))):
        reqs = data.draw(st.permutations(list(range(R))))[: data.draw(st.integers(0, R))]
        segs = []
        for r in reqs:
            room = C - ln[r]
            if room == 0:
                continue
            n = data.draw(st.integers(1, room))
            segs.append((r, 1 if n == 1 and data.draw(st.booleans()) else 0, ln[r], n))
        req, pos, slot, ln2 = O.ring_index_model(R, C, base, ln, segs)
        for r, p, s in zip(req, pos, slot):
            assert s // C == r and s not in owner                       # own region, never a live slot
            owner[s] = (r, p)
        ln = ln2
        if data.draw(st.booleans()) and R > 0:
            r = data.draw(st.integers(0, R - 1))
            base[r], ln[r] = O.ring_reset_model(C, base[r], ln[r], data.draw(st.integers(-1, 3 * C)))
            owner = {s: v for s, v in owner.items() if v[0] != r}


# ------------------------------------------------------------------ P9: values the paper prints for the schedule
def test_p9_steady_schedule_matches_paper_values():
    L_P, K, R = 276, 7, 8                                               # 256 vision + 20 prompt tokens, K = 7
    ln = [0] * R
    base = [0] * R
    appended = {}
    for step in range(40):
        segs = I.steady_schedule(step, L_P, K, R)
        if step >= K - 1:
            assert I.total_rows(segs) == L_P + (K - 1) == 282           # L_Q = L_P + (K-1)
            ctx = [s[2] + s[3] for s in segs[1:]]
            assert ctx == [L_P + s for s in range(1, K)] == list(range(277, 283))   # stage s context L_P+s
            assert I.prediction_rows(segs) == list(range(L_P - 1, L_P + K - 1))      # rows 275..281 (A3)
        pre = segs[0][0]
        base[pre], ln[pre] = O.ring_reset_model(512, base[pre], ln[pre], -1)         # recycle before each prefill
        _, _, _, ln = O.ring_index_model(R, 512, base, ln, segs)                     # must validate every step
        for (r, ph, st_, n) in segs:
            appended.setdefault((r, step - (0 if ph == 0 else st_ - L_P + 1)), []).append((st_, n))
    # every request: 1 prefill + K-1 decodes at contiguous positions, final length L_P + K - 1
    full = [v for k, v in appended.items() if len(v) == K]
    assert len(full) >= 30
    for v in full:
        assert v == [(0, L_P)] + [(L_P + s - 1, 1) for s in range(1, K)]
