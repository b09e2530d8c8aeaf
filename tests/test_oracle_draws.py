"""Pins for the oracle's random draws and threshold (CPU only).

What is pinned and by what:
  * Philox4x32-10            <- the published Random123 known-answer vectors (tests/golden)
  * draw field layout (R11)  <- SURVEY.md's independently computed contract examples (tests/golden)
  * draw -> state map (R9)   <- closed form: state s owns the draws [ceil(s*2^32/q), ceil((s+1)*2^32/q))
  * threshold (R10)          <- closed forms p_c = sqrt(q)/(1+sqrt(q)), q=4 -> 0xAAAAAAAA, K=0, K=inf, ln 2
"""
import math

import numpy as np
import pytest

from oracle import binding as orc


def _hex(x):
    return int(x, 16)


def test_philox_known_answers(golden):
    rows = golden("philox4x32_10_kat.txt")
    assert len(rows) == 3
    for row in rows:
        f = [_hex(v) for v in row.split()]
        assert orc.philox4x32_10(f[0:4], f[4:6]) == tuple(f[6:10])


def test_philox_is_a_bijection_of_the_counter_on_a_sample():
    # a counter-based generator is a keyed bijection: distinct counters -> distinct outputs
    outs = {orc.philox4x32_10((i, 0, 0, 0), (1, 0)) for i in range(4096)}
    assert len(outs) == 4096
    outs2 = {orc.philox4x32_10((0, 0, i, 0), (1, 0)) for i in range(4096)}
    assert len(outs2) == 4096 and len(outs & outs2) == 1   # (0,0,0,0) is shared


def test_contract_examples(golden):
    n = 0
    for row in golden("contract_examples.txt"):
        f = row.split()
        kind = f[0]
        if kind in ("init", "bond", "flip"):
            seed, idx, t = int(f[1], 0), int(f[2], 0), int(f[3], 0)
            want = [None if v == "-" else _hex(v) for v in f[4:8]]
            if kind == "init":
                assert orc.draw_init(seed, idx) == want[0]
            elif kind == "flip":
                assert orc.draw_flip(seed, t, idx) == want[0]
            else:  # idx is the PAIR index: sites 2*idx and 2*idx+1, words (right, down, right, down)
                got = [orc.draw_bond(seed, t, 2 * idx, 0), orc.draw_bond(seed, t, 2 * idx, 1),
                       orc.draw_bond(seed, t, 2 * idx + 1, 0), orc.draw_bond(seed, t, 2 * idx + 1, 1)]
                assert got == want
            n += 1
        elif kind == "initspins":
            q = int(f[1]); want = [int(v) for v in f[2:]]
            got = [orc.state_from_draw(orc.draw_init(1, i), q) for i in range(len(want))]
            assert got == want
            n += 1
        elif kind == "flipstates":
            q = int(f[1]); want = [int(v) for v in f[2:]]
            got = [orc.state_from_draw(orc.draw_flip(1, t, 0), q) for t in range(len(want))]
            assert got == want
            n += 1
    assert n == 24


def test_draws_are_the_stated_words_of_the_pinned_philox():
    # layout consistency against the KAT-pinned block function, on awkward values
    for seed, t, site in [(1, 0, 0), (0xDEADBEEFCAFEF00D, 12345, 0xFFFFFFFF), (7, 0xFFFFFFFF, 2 ** 32 - 2), (3, 5, 65537)]:
        key = (seed & 0xFFFFFFFF, seed >> 32)
        pair = site >> 1
        w = orc.philox4x32_10((pair & 0xFFFFFFFF, pair >> 32, t, 1), key)
        assert orc.draw_bond(seed, t, site, 0) == w[2 * (site & 1)]
        assert orc.draw_bond(seed, t, site, 1) == w[2 * (site & 1) + 1]
        assert orc.draw_flip(seed, t, site) == orc.philox4x32_10((site & 0xFFFFFFFF, site >> 32, t, 2), key)[0]
        assert orc.draw_init(seed, site) == orc.philox4x32_10((site & 0xFFFFFFFF, site >> 32, 0, 0), key)[0]


@pytest.mark.parametrize("q", [2, 3, 4, 5, 10, 255])
def test_state_from_draw_partition(q):
    two32 = 1 << 32
    assert orc.state_from_draw(0, q) == 0
    assert orc.state_from_draw(two32 - 1, q) == q - 1
    for s in range(q):
        lo = -(-s * two32 // q)                 # ceil(s*2^32/q): first draw of state s
        assert orc.state_from_draw(lo, q) == s
        if lo > 0:
            assert orc.state_from_draw(lo - 1, q) == s - 1
    if q == 2:
        for w in (0x7FFFFFFF, 0x80000000, 0x12345678, 0xF0000000):
            assert orc.state_from_draw(w, 2) == w >> 31


@pytest.mark.parametrize("q", [2, 3, 10])
def test_init_states_are_uniform(q):
    n = 60000
    counts = np.bincount([orc.state_from_draw(orc.draw_init(5, i), q) for i in range(n)], minlength=q)
    chi2 = float(((counts - n / q) ** 2 / (n / q)).sum())
    # chi^2 with q-1 dof: mean q-1, sd sqrt(2(q-1)); 6 sd is far outside any plausible fluctuation
    assert chi2 < (q - 1) + 6 * math.sqrt(2 * (q - 1)) + 4


def test_threshold_table(golden):
    for row in golden("thresholds.txt"):
        _, khex, T = row.split()
        assert orc.threshold(float.fromhex(khex)) == int(T)


def test_threshold_closed_forms():
    two32 = 1 << 32
    assert orc.threshold(0.0) == 0
    assert orc.threshold(math.inf) == two32
    assert orc.threshold(math.log(3.0)) == 0xAAAAAAAA          # q = 4: p_c = 2/3
    assert orc.threshold(math.log(2.0)) == 1 << 31             # p = 1/2
    for q in (2, 3, 4, 5, 10, 100):
        K = math.log(1.0 + math.sqrt(q))                       # paper: T_c/J = 1/ln(1+sqrt 2) at q=2
        p_c = math.sqrt(q) / (1.0 + math.sqrt(q))
        assert abs(orc.threshold(K) - p_c * two32) <= 2.0
    assert abs(1.0 / math.log(1.0 + math.sqrt(2.0)) - 1.1346) < 5e-5     # the value the paper prints
    # monotone in K, saturating below 2^32 for any finite K
    ks = np.linspace(0, 30, 301)
    ts = [orc.threshold(float(k)) for k in ks]
    assert all(a <= b for a, b in zip(ts, ts[1:])) and ts[-1] <= two32
    for bad in (-1.0, float("nan"), -math.inf):
        with pytest.raises(orc.OracleError):
            orc.threshold(bad)
