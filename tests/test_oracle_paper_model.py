"""Pins for the oracle's model 4 -- the paper's own agent model (SIII-C, PAPER.md:134-141;
SURVEY.md S8(f)-2; reading A24): mid-price reference (Eq.3), marketable orders,
parity-alternating makers, momentum on mid changes, classes by contiguous index ranges.  No GPU.
"""
import numpy as np
import pytest

from ks_testlib import read_golden
from paper_2606_21784_b200.workloads import paper_params

REC = {n: i for i, n in enumerate(
    ("steps", "n_trades", "sum_vol", "sum_px", "sum_px2", "sum_pxvol", "sum_ret", "sum_ret2",
     "sum_ret3", "sum_ret4", "sub_buy", "sub_sell", "last", "prev", "traj_hash", "n_orders"))}


def test_first_order_by_hand_from_kat1(oracle):
    """tests/golden/paper_model_first_order.txt: agent 0, step 0, market 0, seed 0 -> Philox KAT #1.
    One record per class: noise (half-tick / integer mid, marketable), momentum (rising, falling,
    flat -> coin, half-tick mids, marketable both ways, the threshold itself), maker (never marketable)."""
    seen = set()
    for g in read_golden("paper_model_first_order.txt"):
        cls = g.get("class", ["noise"])[0]
        seen.add(cls)
        A = 100
        p = paper_params(A, 1.0 if cls == "momentum" else 0.0, 1.0 if cls == "maker" else 0.0,
                         delta=int(g["delta"][0]), qmax=int(g["qmax"][0]), half_spread=3, p_mkt=0.0)
        p["paper_pmkt_q16"] = int(g["pmkt_q16"][0])
        mid2 = int(g["mid2"][0])
        prev2 = int(g.get("prev2", g["mid2"])[0])
        got = oracle.gen_orders_paper(p, int(g["L"][0]), mid2, prev2, 0, 0, 0, 0, A)
        assert got == (0 if g["order"][0] == "B" else 1, int(g["order"][1]), int(g["order"][2])), g["name"]
    assert seen == {"noise", "momentum", "maker"}


def test_momentum_follows_the_mid_not_the_last_price(oracle):
    """PAPER.md:139 through the run loop: ret_t = sgn(mid_t - mid_{t-1}) with mid from Eq.3 on the
    RESTING book, p = round(mid + side).  A momentum-only population on an injected book whose mid
    (12.5) is far from the last price (30 resp. 5): every order of the step lands on ONE tick, and
    that tick is round(mid -/+ 1), not last -/+ 1.  Worked by hand:
      market 0: last 30 -> f[13] = 60 (doubled opening mid); bb 10, ba 15 -> mid2 25 < 60 -> all SELL
                at round(12.5 - 1) = round(11.5) = 12; best bid 10 < 12: no trade
      market 1: last 5  -> f[13] = 10; mid2 25 > 10 -> all BUY at round(12.5 + 1) = round(13.5) = 14;
                best ask 15 > 14: no trade"""
    L, A = 64, 50
    p = paper_params(A, 1.0, 0.0, qmax=5, p_mkt=0.0)
    for init, side, tick in ((30, 1, 12), (5, 0, 14)):
        books = np.zeros((1, 2, L), dtype=np.int32)
        books[0, 0, 10] = 7; books[0, 0, 4] = 9; books[0, 1, 15] = 3; books[0, 1, 40] = 1
        _, recs = oracle.init_state(1, L, init, model=4)
        assert recs[0, REC["prev"]] == 2 * init
        b, r = oracle.run_markets(dict(p, init_price=init), L, A, 3, [0], 1, books, recs)
        d = b.astype(np.int64) - books
        assert set(np.flatnonzero(d[0, side])) == {tick} and not d[0, 1 - side].any()
        assert r[0, REC["n_trades"]] == 0 and r[0, REC["prev"]] == 25 and r[0, REC["last"]] == init
        assert d[0, side, tick] == r[0, REC["sub_sell" if side else "sub_buy"]]
    # second step of market 0: the book now rests bb 10 / ba 12 -> mid2 22 < 25 -> SELL at
    # round(11 - 1) = 10, which crosses the 7 lots bid at tick 10: p* = 10, Vmax = 7
    books = np.zeros((1, 2, L), dtype=np.int32)
    books[0, 0, 10] = 7; books[0, 0, 4] = 9; books[0, 1, 15] = 3; books[0, 1, 40] = 1
    _, recs = oracle.init_state(1, L, 30, model=4)
    b, r = oracle.run_markets(dict(p, init_price=30), L, A, 3, [0], 2, books, recs)
    assert r[0, REC["prev"]] == 22 and r[0, REC["last"]] == 10 and r[0, REC["sum_vol"]] == 7 and b[0, 0, 10] == 0


def test_mid_price_retrieval_eq3(oracle):
    """Eq.3 seen through a makers-only population: every order sits at
    round(mid -/+ h), so the ticks that gain depth reveal the mid the oracle used."""
    L, A, h = 64, 40, 2
    p = paper_params(A, 0.0, 1.0, half_spread=h, qmax=5)             # all makers
    books = np.zeros((3, 2, L), dtype=np.int32)
    books[0, 0, 10] = 7; books[0, 0, 4] = 9; books[0, 1, 15] = 3; books[0, 1, 40] = 1   # bb = 10, ba = 15
    books[1, 0, 20] = 5                                                                 # one-sided
    # market 2: empty
    _, recs = oracle.init_state(3, L, 30, model=4)
    b, r = oracle.run_markets(p, L, A, 1, [0, 1, 2], 1, books, recs)
    d = b.astype(np.int64) - books
    # market 0: mid2 = 25 -> bid at round(12.5 - 2) = floor(10.5 + .5) = 11, ask at round(14.5) = 15
    assert set(np.flatnonzero(d[0, 0] > 0)) == {11} and set(np.flatnonzero(d[0, 1] > 0)) <= {15}
    assert r[0, REC["prev"]] == 25
    # markets 1, 2: no two-sided book -> mid = last = 30 -> bids at 28, asks at 32; nothing crosses
    for i in (1, 2):
        assert set(np.flatnonzero(d[i, 0] > 0)) == {28} and set(np.flatnonzero(d[i, 1] > 0)) == {32}
        assert r[i, REC["prev"]] == 60 and r[i, REC["n_trades"]] == 0
    # maker parity: agent a buys at step t iff (a + t) even -> at t = 0 the even agents bid
    sides = [oracle.gen_orders_paper(p, L, 60, 60, 1, 0, t, a, A)[0] for t in (0, 1) for a in range(4)]
    assert sides == [0, 1, 0, 1, 1, 0, 1, 0]


def test_rules_against_exact_integer_restatement(oracle):
    """Every class, signs of the mid change, both parities of mid2, grid edges (negative and
    beyond-grid prices before the clamp): round-half-up is floor((m2 + 1) / 2) in exact integers."""
    L, A = 128, 90
    p = paper_params(A, 0.3, 0.2, delta=20, qmax=10, half_spread=3, p_mkt=0.25)
    n_mom, n_mk = p["paper_n_mom"], p["paper_n_maker"]
    n_noise = A - n_mom - n_mk
    for mid2, prev2 in [(127, 127), (128, 120), (3, 9), (0, 0), (253, 250), (254, 254), (37, 38)]:
        for a in range(A):
            for t in (0, 5):
                w = [int(x) for x in oracle.philox4x32_10([a, t, 9, 0], [11, 0])]
                coin, mkt = w[0] >> 31, (w[3] >> 16) < p["paper_pmkt_q16"]
                if a < n_noise:
                    buy, m2, qm = coin, mid2 + 2 * (((w[1] * 41) >> 32) - 20), 10
                elif a < n_noise + n_mom:
                    buy = 1 if mid2 > prev2 else (0 if mid2 < prev2 else coin)
                    m2, qm = mid2 + (2 if buy else -2), 10
                else:
                    buy, mkt = int((a + t) % 2 == 0), False
                    m2, qm = mid2 + (-6 if buy else 6), 10
                tick = min(max((m2 + 1) // 2, 0), L - 1)           # Python // floors
                if mkt:
                    tick = L - 1 if buy else 0
                q = 1 + ((w[2] * qm) >> 32)
                assert oracle.gen_orders_paper(p, L, mid2, prev2, 11, 9, t, a, A) == (0 if buy else 1, tick, q)


def test_marketable_fraction(oracle):
    L, A = 256, 1000
    for pm in (0.0, 0.05, 0.5, 1.0):
        p = paper_params(A, 0.0, 0.0, p_mkt=pm)
        n = sum(oracle.gen_orders_paper(p, L, 256, 256, 3, 1, t, a, A)[1] in (0, L - 1)
                for t in range(20) for a in range(A))
        exp = 20 * A * pm
        assert abs(n - exp) <= 4.5 * np.sqrt(max(exp * (1 - pm), 1e-9)) + (0 if pm in (0.0, 1.0) else 1)


@pytest.mark.parametrize("alpha_mom", [0.0, 0.15, 0.6])
def test_per_step_invariants_and_state_carry(oracle, alpha_mom):
    L, A, S, seed, ids = 128, 200, 60, 5, [0, 3]
    p = paper_params(A, alpha_mom)
    books, recs = oracle.init_state(len(ids), L, -1, model=4)
    assert (recs[:, REC["prev"]] == 2 * recs[:, REC["last"]]).all()
    for t in range(S):
        before = books.copy()
        books, recs = oracle.run_markets(p, L, A, seed, ids, 1, books, recs)
        for i in range(len(ids)):
            bid, ask = books[i, 0].astype(np.int64), books[i, 1].astype(np.int64)
            assert (bid >= 0).all() and (ask >= 0).all()
            assert recs[i, REC["sub_buy"]] == recs[i, REC["sum_vol"]] + bid.sum()
            assert recs[i, REC["sub_sell"]] == recs[i, REC["sum_vol"]] + ask.sum()
            assert recs[i, REC["n_orders"]] == (t + 1) * A
            if bid.any() and ask.any():
                assert np.flatnonzero(bid).max() < np.flatnonzero(ask).min()
            # f[13] = doubled mid of the book the step STARTED from (Eq.3)
            b0, a0 = before[i, 0], before[i, 1]
            exp_mid2 = (np.flatnonzero(b0).max() + np.flatnonzero(a0).min()) if (b0.any() and a0.any()) else None
            if exp_mid2 is not None:
                assert recs[i, REC["prev"]] == exp_mid2
    b1, r1 = oracle.run_markets(p, L, A, seed, ids, 25)
    b1, r1 = oracle.run_markets(p, L, A, seed, ids, S - 25, b1, r1)
    assert np.array_equal(b1, books) and np.array_equal(r1, recs)
