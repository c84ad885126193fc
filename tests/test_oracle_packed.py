"""Pins for the oracle's PACKED4 draw contract (models 2 and 3, DESIGN.md
reading A22): one Philox block per four consecutive agents, every draw out of one 32-bit word by
successive multiply-extract.  No GPU.

What fixes it, other than the oracle itself:
  * Philox known-answer vector #1 -> the first four orders of C1 under PACKED4, derived by hand
    with exact integers (tests/golden/packed4_first_orders.txt);
  * the mixed-radix identity: with N = n*qmax*2 and J = floor(w*N / 2^32) in Python big integers,
    the draws are the digits of J (coin = J mod 2, q-1 = (J div 2) mod qmax, o_index = J div 2qmax)
    -- the sequential hi/lo extraction of the C code must agree with it for every word;
  * which block and which word an agent reads (agents 4b..4b+3 <-> words 0..3 of block b, block
    counter = (b, step, market, 0)), checked against the KAT-pinned Philox routine;
  * uniformity (chi-square) of side, offset and quantity, and independence of the three digits;
  * the per-step trajectory invariants of the literal contract, which do not depend on how orders
    are drawn.
"""
import numpy as np
import pytest

from ks_testlib import read_golden
from paper_2606_21784_b200.workloads import mix3_params, packed4, zi_params

REC = {n: i for i, n in enumerate(
    ("steps", "n_trades", "sum_vol", "sum_px", "sum_px2", "sum_pxvol", "sum_ret", "sum_ret2",
     "sum_ret3", "sum_ret4", "sub_buy", "sub_sell", "last", "prev", "traj_hash", "n_orders"))}


def _digits(w, n, qmax):
    """(o_index, q, coin) of word w by exact integer arithmetic."""
    J = (int(w) * (n * qmax * 2)) >> 32
    return J // (2 * qmax), 1 + (J // 2) % qmax, J % 2


def _word(oracle, seed, m, t, a):
    key = [seed & 0xffffffff, seed >> 32]
    return int(oracle.philox4x32_10([a >> 2, t, m, 0], key)[a & 3])


def test_first_four_orders_of_c1_by_hand(oracle):
    g = read_golden("packed4_first_orders.txt")[0]
    p = packed4(zi_params(int(g["delta"][0]), int(g["qmax"][0])))
    L, last = int(g["L"][0]), int(g["last"][0])
    exp = [(0 if g["orders"][3 * i] == "B" else 1, int(g["orders"][3 * i + 1]), int(g["orders"][3 * i + 2]))
           for i in range(4)]
    got = [oracle.gen_orders(p, L, last, last, 0, 0, 0, a)[0] for a in range(4)]
    assert got == exp


def test_noise_draws_are_the_mixed_radix_digits_of_one_word(oracle):
    L, last = 1024, 500
    for (delta, qmax) in [(8, 10), (32, 100), (64, 50), (0, 1), (300, 1 << 20)]:
        p = packed4(zi_params(delta, qmax))
        n = 2 * delta + 1
        for seed, m, t in [(0, 0, 0), (3, 65535, 999), ((7 << 32) | 5, 2 ** 32 - 1, 2 ** 32 - 1)]:
            for a in list(range(0, 41)) + [4095, 4096, 4097, 2 ** 32 - 1]:
                oi, q, coin = _digits(_word(oracle, seed, m, t, a), n, qmax)
                o = oi - delta
                tick = min(max(last - o, 0), L - 1) if coin else min(max(last + o, 0), L - 1)
                assert oracle.gen_orders(p, L, last, last, seed, m, t, a) == [(0 if coin else 1, tick, q)]


def test_mix3_packed_rules(oracle):
    p = packed4(mix3_params())
    L = 4096
    for last, prev in [(2000, 2000), (2000, 1999), (2000, 2003), (3, 3), (4093, 4090)]:
        for a in range(0, 60):
            w = _word(oracle, 4, 17, 5, a)
            got = oracle.gen_orders(p, L, last, prev, 4, 17, 5, a)
            cl = lambda x: min(max(x, 0), L - 1)
            if a % 3 == 0:
                oi, q, coin = _digits(w, 129, 50)
                o = oi - 64
                assert got == [(0, cl(last - o), q)] if coin else got == [(1, cl(last + o), q)]
            elif a % 3 == 1:
                s = 1 + ((w * 4) >> 32)
                assert got == [(0, cl(last - s), 20), (1, cl(last + s), 20)]
            else:
                oi, q, coin = _digits(w, 9, 50)
                buy = 1 if last > prev else (0 if last < prev else coin)
                assert got == [(0, cl(last + oi), q)] if buy else got == [(1, cl(last - oi), q)]


def test_block_and_word_assignment(oracle):
    """Agents 4b..4b+3 read words 0..3 of ONE block keyed by (b, step, market, seed); swapping
    the roles of agent block / step / market, or the key halves, changes the orders."""
    p = packed4(zi_params(100, 1000))
    L, last = 4096, 2048
    base = [oracle.gen_orders(p, L, last, last, 9, 5, 6, a) for a in range(28, 32)]
    assert len({tuple(o[0]) for o in base}) == 4                      # four different words
    for other in [dict(seed=9, m=6, t=5), dict(seed=9 << 32, m=5, t=6), dict(seed=9, m=5, t=7)]:
        alt = [oracle.gen_orders(p, L, last, last, other["seed"], other["m"], other["t"], a) for a in range(28, 32)]
        assert alt != base
    # the literal contract (model 0) draws something else for the same agents
    lit = [oracle.gen_orders(zi_params(100, 1000), L, last, last, 9, 5, 6, a) for a in range(28, 32)]
    assert lit != base


def test_packed_noise_distributions(oracle):
    """chi-square uniformity of side (2), offset (2*8+1) and quantity (10), and of the joint
    (side, quantity) table, over 60000 draws."""
    delta, qmax = 8, 10
    p = packed4(zi_params(delta, qmax))
    L, last, N = 256, 128, 60000
    side = np.zeros(2); off = np.zeros(2 * delta + 1); qty = np.zeros(qmax); joint = np.zeros((2, qmax))
    for a in range(N):
        (s, tick, q), = oracle.gen_orders(p, L, last, last, 1, a % 7, a // 977, a)
        o = (last - tick) if s == 0 else (tick - last)
        side[s] += 1; off[o + delta] += 1; qty[q - 1] += 1; joint[s, q - 1] += 1
    def chi2(c):
        e = c.sum() / c.size
        return float(((c - e) ** 2 / e).sum())
    assert chi2(side) < 10.8            # 1 dof, p = 0.001
    assert chi2(off) < 39.3             # 16 dof
    assert chi2(qty) < 27.9             # 9 dof
    assert chi2(joint) < 43.8           # 19 dof


@pytest.mark.parametrize("model", ["zi", "mix3"])
def test_per_step_invariants_packed(oracle, model):
    """Conservation, non-negativity, uncrossed book after every step, price fields (as for the
    literal contract: these do not depend on how the orders are drawn)."""
    if model == "zi":
        L, A, S, seed, p, ids = 128, 510, 50, 2, packed4(zi_params(8, 10)), [0, 31]   # A % 4 != 0
    else:
        L, A, S, seed, p, ids = 256, 301, 50, 4, packed4(mix3_params()), [0, 9]
    n_makers = sum(1 for a in range(A) if model == "mix3" and a % 3 == 1)
    books, recs = oracle.init_state(len(ids), L, -1)
    for t in range(S):
        prev_recs = recs.copy()
        books, recs = oracle.run_markets(p, L, A, seed, ids, 1, books, recs)
        for i in range(len(ids)):
            r, q = recs[i], prev_recs[i]
            bid, ask = books[i, 0].astype(np.int64), books[i, 1].astype(np.int64)
            assert (bid >= 0).all() and (ask >= 0).all()
            assert r[REC["sub_buy"]] == r[REC["sum_vol"]] + bid.sum()
            assert r[REC["sub_sell"]] == r[REC["sum_vol"]] + ask.sum()
            assert r[REC["n_orders"]] == (t + 1) * (A + n_makers)
            if bid.any() and ask.any():
                assert np.flatnonzero(bid).max() < np.flatnonzero(ask).min()
            assert r[REC["prev"]] == q[REC["last"]]
    # split runs carry the state
    b1, r1 = oracle.run_markets(p, L, A, seed, ids, 20)
    b1, r1 = oracle.run_markets(p, L, A, seed, ids, 30, b1, r1)
    assert np.array_equal(b1, books) and np.array_equal(r1, recs)
