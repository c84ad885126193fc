"""Pins for the CPU oracle (oracle/ks_oracle.c) against things OTHER than itself: published
known-answer vectors, the paper's worked example, hand-worked cases, a literal O(L^2) evaluation
of Eq.1-2, greedy lot-by-lot matching, closed forms, per-step invariants, distribution checks and
a numpy return series.  No GPU.  Each test names the passage it pins."""
import numpy as np
import pytest

from ks_testlib import brute_force_price, greedy_match, ints, read_golden
from paper_2606_21784_b200.workloads import CONFIGS, mix3_params, zi_params


# ---------------------------------------------------------------- Philox4x32-10 (north_star (1))
def test_philox_known_answers(oracle):
    recs = read_golden("philox_kat.txt")
    assert len(recs) == 3
    for r in recs:
        ctr = [int(x, 16) for x in r["ctr"]]
        key = [int(x, 16) for x in r["key"]]
        out = [int(x, 16) for x in r["out"]]
        got = oracle.philox4x32_10(ctr, key)
        assert [int(x) for x in got] == out


def test_first_order_of_c1_by_hand(oracle):
    """Counter/key layout and word->field mapping: with seed 0, market 0, step 0, agent 0 the
    Philox block is KAT #1, so by hand: w0 top bit 0 -> SELL; mulhi(0xe169c58d, 17) = 14 -> o = +6
    -> tick 32+6 = 38; mulhi(0xbc57ac4c, 10) = 7 -> qty 8."""
    assert (0xe169c58d * 17) >> 32 == 14 and (0xbc57ac4c * 10) >> 32 == 7
    c = CONFIGS["C1"]
    assert oracle.gen_orders(c.params, c.L, 32, 32, 0, 0, 0, 0) == [(1, 38, 8)]


def test_counter_layout_is_agent_step_market(oracle):
    """ctr = (agent, step, market, 0), key = (seed lo, seed hi): permuting the roles must change
    the draw, and the draw must equal the rule applied to the block of exactly that counter."""
    p = zi_params(8, 10)
    L, last = 64, 32
    for (seed, m, t, a) in [(0x1234567890ABCDEF, 3, 5, 7), (1, 1000, 999, 4095), (2**64 - 1, 7, 0, 1)]:
        w = [int(x) for x in oracle.philox4x32_10([a, t, m, 0], [seed & 0xffffffff, seed >> 32])]
        buy = w[0] >> 31
        o = ((w[1] * 17) >> 32) - 8
        q = 1 + ((w[2] * 10) >> 32)
        tick = min(max(last - o if buy else last + o, 0), L - 1)
        assert oracle.gen_orders(p, L, last, last, seed, m, t, a) == [(0 if buy else 1, tick, q)]
    # swapping agent and market gives a different block
    assert oracle.gen_orders(p, L, last, last, 9, 1, 0, 2) != oracle.gen_orders(p, L, last, last, 9, 2, 0, 1) \
        or oracle.gen_orders(p, L, last, last, 9, 1, 0, 3) != oracle.gen_orders(p, L, last, last, 9, 3, 0, 1)


def _chi2(counts, expected):
    counts = np.asarray(counts, dtype=np.float64)
    return float(((counts - expected) ** 2 / expected).sum())


def test_noise_rule_distributions(oracle):
    """side ~ 50 %, offsets uniform over 2D+1 values, qty uniform over 1..qmax;
    chi-square on 2*10^5 draws, thresholds far in the tail (p < 1e-6)."""
    p = zi_params(16, 100)
    L, last, n = 256, 128, 200_000
    side = np.zeros(2); off = np.zeros(33); qty = np.zeros(100)
    for a in range(n):
        (s, tick, q), = oracle.gen_orders(p, L, last, last, 1, a % 7, a // 1024, a)
        side[s] += 1
        o = (tick - last) if s == 1 else (last - tick)      # bid offsets mirrored (A11)
        off[o + 16] += 1
        qty[q - 1] += 1
    assert _chi2(side, n / 2) < 30          # 1 dof
    assert _chi2(off, n / 33) < 90          # 32 dof
    assert _chi2(qty, n / 100) < 190        # 99 dof


def test_clamp_piles_on_edges(oracle):
    """Out-of-grid prices are clamped to [0, L-1] (A15)."""
    p = zi_params(8, 10)
    for a in range(200):
        for last in (0, 63):
            (s, tick, q), = oracle.gen_orders(p, 64, last, last, 5, 0, 0, a)
            assert 0 <= tick <= 63 and abs(tick - last) <= 8 and 1 <= q <= 10


def test_mix3_rules(oracle):
    """Type by a mod 3 (A14); maker posts both sides at last -/+ s, s in 1..4, qty 20 (A13);
    momentum follows sign(last - prev), tie -> w0 bit, offset in [0,8] toward the aggressive
    side (A12)."""
    p = mix3_params()
    L = 4096
    seen_s = set()
    for a in range(0, 3000, 3):
        o = oracle.gen_orders(p, L, 2048, 2048, 4, 1, 2, a)
        assert len(o) == 1 and abs(o[0][1] - 2048) <= 64 and 1 <= o[0][2] <= 50
        mk = oracle.gen_orders(p, L, 2048, 2040, 4, 1, 2, a + 1)
        assert len(mk) == 2 and mk[0][0] == 0 and mk[1][0] == 1 and mk[0][2] == mk[1][2] == 20
        s = 2048 - mk[0][1]
        assert mk[1][1] - 2048 == s and 1 <= s <= 4
        seen_s.add(s)
        w = [int(x) for x in oracle.philox4x32_10([a + 2, 2, 1, 0], [4, 0])]
        up, = oracle.gen_orders(p, L, 2048, 2040, 4, 1, 2, a + 2)      # price rose -> buy above
        dn, = oracle.gen_orders(p, L, 2048, 2050, 4, 1, 2, a + 2)      # price fell -> sell below
        tie, = oracle.gen_orders(p, L, 2048, 2048, 4, 1, 2, a + 2)
        assert up[0] == 0 and 0 <= up[1] - 2048 <= 8 and 1 <= up[2] <= 50
        assert dn[0] == 1 and 0 <= 2048 - dn[1] <= 8 and dn[2] == up[2]
        assert up[1] - 2048 == 2048 - dn[1] == (w[1] * 9) >> 32
        assert tie[0] == (0 if (w[0] >> 31) else 1)
    assert seen_s == {1, 2, 3, 4}
    # edge clamp of the maker
    mk = oracle.gen_orders(p, L, 0, 0, 4, 1, 2, 1)
    assert mk[0][1] == 0 and 1 <= mk[1][1] <= 4


# ---------------------------------------------------------------- clearing (Eq.1-2, SIV-C)
def _check_case(oracle, r):
    res = oracle.clear_step(ints(r, "BUY"), ints(r, "SELL"))
    assert list(res["D"]) == list(ints(r, "D"))
    assert list(res["S"]) == list(ints(r, "S"))
    assert list(res["V"]) == list(ints(r, "V"))
    assert res["pstar"] == int(r["pstar"][0])
    assert res["vmax"] == int(r["vmax"][0])
    assert list(res["new_bid"]) == list(ints(r, "new_bid"))
    assert list(res["new_ask"]) == list(ints(r, "new_ask"))


def test_paper_worked_example(oracle):
    """PAPER.md:315-354, Eq.11-18: every intermediate the paper prints."""
    recs = read_golden("paper_worked_example.txt")
    assert len(recs) == 1
    _check_case(oracle, recs[0])


def test_hand_worked_cases(oracle):
    recs = read_golden("hand_cases.txt")
    assert len(recs) == 6
    for r in recs:
        _check_case(oracle, r)


def test_closed_form_single_bid_single_ask(oracle):
    """One bid x@b and one ask y@a: a <= b -> V = min(x, y) at p* = a (lowest tick of the plateau
    [a, b]); a > b -> no trade."""
    L = 7
    for b in range(L):
        for a in range(L):
            for x, y in [(5, 3), (3, 5), (4, 4)]:
                bid = np.zeros(L, np.int64); ask = np.zeros(L, np.int64)
                bid[b] = x; ask[a] = y
                res = oracle.clear_step(bid, ask)
                if a <= b:
                    assert (res["pstar"], res["vmax"]) == (a, min(x, y))
                    assert res["new_bid"][b] == x - min(x, y) and res["new_ask"][a] == y - min(x, y)
                else:
                    assert (res["pstar"], res["vmax"]) == (-1, 0)
                    assert res["new_bid"][b] == x and res["new_ask"][a] == y


@pytest.mark.parametrize("L", [1, 2, 3, 5, 8])
def test_brute_force_and_greedy_on_random_tiny_books(oracle, L):
    """Literal O(L^2) Eq.1-2 gives the same D, S, p*, Vmax; lot-by-lot price-priority matching
    gives the same volume and the same residual arrays (reading A5)."""
    rng = np.random.default_rng(100 + L)
    for _ in range(1500):
        fill = rng.random()
        bid = rng.integers(0, 7, L) * (rng.random(L) < fill)
        ask = rng.integers(0, 7, L) * (rng.random(L) < fill)
        res = oracle.clear_step(bid, ask)
        ps, vm, D, S = brute_force_price(bid, ask)
        assert (res["pstar"], res["vmax"]) == (ps, vm)
        assert list(res["D"]) == D and list(res["S"]) == S
        vol, nb, na = greedy_match(bid, ask)
        assert vol == vm
        assert list(res["new_bid"]) == list(nb) and list(res["new_ask"]) == list(na)


def test_clearing_invariants_random_books(oracle):
    """V is unimodal; after clearing the book is uncrossed; residual <= combined per tick;
    min ask tick <= p* <= max bid tick of the combined book."""
    rng = np.random.default_rng(7)
    for _ in range(300):
        L = int(rng.integers(2, 40))
        bid = rng.integers(0, 50, L) * (rng.random(L) < 0.4)
        ask = rng.integers(0, 50, L) * (rng.random(L) < 0.4)
        res = oracle.clear_step(bid, ask)
        V = res["V"]
        k = int(np.argmax(V))
        assert np.all(np.diff(V[:k + 1]) >= 0) and np.all(np.diff(V[k:]) <= 0)
        nb, na = res["new_bid"], res["new_ask"]
        assert np.all(nb >= 0) and np.all(na >= 0) and np.all(nb <= bid) and np.all(na <= ask)
        assert (bid - nb).sum() == (ask - na).sum() == res["vmax"]
        if nb.any() and na.any():
            assert np.flatnonzero(nb).max() < np.flatnonzero(na).min()
        if res["vmax"] > 0:
            assert np.flatnonzero(ask).min() <= res["pstar"] <= np.flatnonzero(bid).max()
