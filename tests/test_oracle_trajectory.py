"""Whole-trajectory pins for the oracle: per-step invariants, state carry, the surveyor's
independent scratch-simulator values, the derived fp64 statistics against a numpy return series,
and the trajectory hash against its definition.  No GPU."""
import numpy as np
import pytest

from ks_testlib import read_golden
from paper_2606_21784_b200.workloads import CONFIGS, mix3_params, zi_params, sampled_markets, shard_markets

REC = {n: i for i, n in enumerate(
    ("steps", "n_trades", "sum_vol", "sum_px", "sum_px2", "sum_pxvol", "sum_ret", "sum_ret2",
     "sum_ret3", "sum_ret4", "sub_buy", "sub_sell", "last", "prev", "traj_hash", "n_orders"))}


def _params_of(model_words):
    if model_words[0] == "zi":
        return zi_params(int(model_words[1]), int(model_words[2]))
    return mix3_params()


def test_record_layout_names(oracle):
    assert {n: i for i, n in enumerate(oracle.REC_FIELDS)} == REC


@pytest.mark.parametrize("case", ["C1", "C3-short", "C2-short", "MIX3-small"])
def test_per_step_invariants(oracle, case):
    """north_star invariants on every step: executed buy volume == executed sell volume (asserted
    inside the oracle, code -2), quantity conserved across orders, fills and residual book
    (submitted = filled + resting per side), volume never negative; plus: the book is uncrossed
    after every step, and the record's price fields follow the step rule (A4)."""
    if case == "C1":
        c = CONFIGS["C1"]; L, A, S, seed, p, ids = c.L, c.A, c.S, c.seed, c.params, [0]
    elif case == "C3-short":
        c = CONFIGS["C3"]; L, A, S, seed, p, ids = c.L, c.A, 60, c.seed, c.params, [0, 31]
    elif case == "C2-short":
        c = CONFIGS["C2"]; L, A, S, seed, p, ids = c.L, c.A, 25, c.seed, c.params, [5, 1023]
    else:
        L, A, S, seed, p, ids = 256, 300, 80, 4, mix3_params(), [0, 9]
    books, recs = oracle.init_state(len(ids), L, -1)
    n_makers = sum(1 for a in range(A) if p["model"] == 1 and a % 3 == 1)
    for t in range(S):
        prev_recs = recs.copy()
        books, recs = oracle.run_markets(p, L, A, seed, ids, 1, books, recs)
        for i in range(len(ids)):
            r, q = recs[i], prev_recs[i]
            bid, ask = books[i, 0].astype(np.int64), books[i, 1].astype(np.int64)
            assert (bid >= 0).all() and (ask >= 0).all()
            assert r[REC["sub_buy"]] == r[REC["sum_vol"]] + bid.sum()
            assert r[REC["sub_sell"]] == r[REC["sum_vol"]] + ask.sum()
            assert r[REC["steps"]] == t + 1 and r[REC["n_orders"]] == (t + 1) * (A + n_makers)
            if bid.any() and ask.any():
                assert np.flatnonzero(bid).max() < np.flatnonzero(ask).min()
            assert r[REC["prev"]] == q[REC["last"]]
            traded = r[REC["n_trades"]] - q[REC["n_trades"]]
            assert traded in (0, 1)
            if traded:
                px = r[REC["sum_px"]] - q[REC["sum_px"]]
                assert r[REC["last"]] == px and r[REC["sum_vol"]] > q[REC["sum_vol"]]
                assert r[REC["sum_px2"]] - q[REC["sum_px2"]] == px * px
                assert r[REC["sum_pxvol"]] - q[REC["sum_pxvol"]] == px * (r[REC["sum_vol"]] - q[REC["sum_vol"]])
            else:
                assert r[REC["last"]] == q[REC["last"]] and r[REC["sum_vol"]] == q[REC["sum_vol"]]


def test_state_carry_split_run(oracle):
    """run(S1); run(S2) == run(S1+S2) (step index is global: SURVEY.md S8(b) 'State carry')."""
    p = mix3_params()
    ids = [0, 3, 17]
    b1, r1 = oracle.run_markets(p, 128, 90, 11, ids, 37)
    b1, r1 = oracle.run_markets(p, 128, 90, 11, ids, 23, b1, r1)
    b2, r2 = oracle.run_markets(p, 128, 90, 11, ids, 60)
    assert np.array_equal(b1, b2) and np.array_equal(r1, r2)


def test_markets_are_independent_and_keyed_by_global_id(oracle):
    """A market's trajectory depends on its global id only (S8(e)): running ids one by one, in
    any order or sharded, gives the same rows."""
    c = CONFIGS["C2"]
    ids = np.array([7, 1000, 3, 512], dtype=np.uint32)
    b, r = oracle.run_markets(c.params, c.L, c.A, c.seed, ids, 12)
    for k in (2, 0, 3, 1):
        bk, rk = oracle.run_markets(c.params, c.L, c.A, c.seed, ids[k:k + 1], 12)
        assert np.array_equal(bk[0], b[k]) and np.array_equal(rk[0], r[k])
    assert not np.array_equal(b[0], b[1])
    covered = []
    for rank in range(3):
        base, cnt = shard_markets(10, rank, 3)
        covered += list(range(base, base + cnt))
    assert covered == list(range(10))


def test_no_agents_books_only_clear(oracle):
    """A = 0: the resting book is cleared as it stands (used to push the paper's worked example
    through the library); a second step finds an uncrossed book and does nothing."""
    ex = read_golden("paper_worked_example.txt")[0]
    L = 32
    books, recs = oracle.init_state(1, L, -1)
    books[0, 0, 10:15] = [int(x) for x in ex["BUY"]]
    books[0, 1, 10:15] = [int(x) for x in ex["SELL"]]
    b, r = oracle.run_markets(zi_params(1, 1), L, 0, 0, [0], 1, books, recs)
    assert list(b[0, 0, 10:15]) == [int(x) for x in ex["new_bid"]]
    assert list(b[0, 1, 10:15]) == [int(x) for x in ex["new_ask"]]
    assert r[0, REC["last"]] == 12 and r[0, REC["sum_vol"]] == 10 and r[0, REC["prev"]] == 16
    b2, r2 = oracle.run_markets(zi_params(1, 1), L, 0, 0, [0], 1, b, r)
    assert np.array_equal(b2, b) and r2[0, REC["n_trades"]] == 1 and r2[0, REC["steps"]] == 2
    assert r2[0, REC["prev"]] == 12 and r2[0, REC["last"]] == 12


def test_survey_scratch_simulator_crosscheck(oracle):
    """SURVEY.md Appendix B values (independent implementation of the same contract)."""
    for g in read_golden("survey_crosscheck.txt"):
        L, A, S, seed, m = (int(g[k][0]) for k in ("L", "A", "S", "seed", "market"))
        p = _params_of(g["model"])
        b, r = oracle.run_markets(p, L, A, seed, [m], S)
        for k in ("n_trades", "sum_vol", "sum_px", "sum_px2", "sum_pxvol", "sum_ret", "sum_ret2",
                  "sum_ret3", "sum_ret4", "sub_buy", "sub_sell", "last", "prev", "n_orders"):
            if k in g:
                assert int(r[0, REC[k]]) == int(g[k][0]), (g["name"], k)
        assert int(r[0, REC["traj_hash"]]) & (2**64 - 1) == int(g["traj_hash"][0], 16), g["name"]
        if "sum_bid" in g:
            assert int(b[0, 0].sum()) == int(g["sum_bid"][0]) and int(b[0, 1].sum()) == int(g["sum_ask"][0])
        if "best_bid" in g:
            assert np.flatnonzero(b[0, 0]).max() == int(g["best_bid"][0])
            assert np.flatnonzero(b[0, 1]).min() == int(g["best_ask"][0])
        if "first_orders" in g:
            w = g["first_orders"]
            exp = [(0 if w[3 * i] == "B" else 1, int(w[3 * i + 1]), int(w[3 * i + 2])) for i in range(4)]
            got = [oracle.gen_orders(p, L, L // 2, L // 2, seed, m, 0, a)[0] for a in range(4)]
            assert got == exp


def test_traj_hash_and_derived_statistics_against_numpy_series(oracle):
    """Step the oracle one step at a time, rebuild the (p*, V) and return series in Python, and
    evaluate (a) the FNV-style trajectory hash from its definition and (b) mean / variance /
    excess kurtosis of the returns with numpy, against the record and ko_derived."""
    p = mix3_params()
    L, A, S, seed = 128, 150, 300, 21
    books, recs = oracle.init_state(1, L, -1)
    h = 0xcbf29ce484222325
    rets, pxs, vols = [], [], []
    for t in range(S):
        before = recs[0].copy()
        books, recs = oracle.run_markets(p, L, A, seed, [0], 1, books, recs)
        v = int(recs[0, REC["sum_vol"]] - before[REC["sum_vol"]])
        traded = int(recs[0, REC["n_trades"]] - before[REC["n_trades"]])
        x = ((v << 16) | int(recs[0, REC["last"]])) if traded else 0xFFFF
        h = ((h ^ x) * 0x100000001b3) & (2**64 - 1)
        rets.append(int(recs[0, REC["last"]] - before[REC["last"]]))
        if traded:
            pxs.append(int(recs[0, REC["last"]])); vols.append(v)
    assert int(recs[0, REC["traj_hash"]]) & (2**64 - 1) == h
    r = np.array(rets, dtype=np.float64)
    assert len(set(rets)) > 2, "test needs a moving price"
    d = oracle.derived(recs[0])
    exp = [np.mean(pxs), np.dot(pxs, vols) / np.sum(vols), np.sum(vols) / S, r.mean(), r.var(),
           ((r - r.mean()) ** 4).mean() / r.var() ** 2 - 3.0]
    assert np.allclose(d, exp, rtol=1e-9, atol=0)
    assert recs[0, REC["sum_ret3"]] == int((np.array(rets) ** 3).sum())
    assert recs[0, REC["sum_ret4"]] == int((np.array(rets) ** 4).sum())


def test_sampled_markets_recipe():
    """ids = {0, M-1} + SplitMix64-driven distinct draws; SplitMix64 pinned by its first outputs
    from state 0 (e220a8397b1dcdaf, 6e789e6aa1b965f4, 06c45d188009454f -- SURVEY.md Appendix A)."""
    from paper_2606_21784_b200.workloads import _splitmix64_stream
    g = _splitmix64_stream(0)
    assert [next(g) for _ in range(3)] == [0xe220a8397b1dcdaf, 0x6e789e6aa1b965f4, 0x06c45d188009454f]
    ids = sampled_markets(65536, 3, 64)
    assert len(ids) == 64 and len(set(ids.tolist())) == 64 and ids[0] == 0 and ids[1] == 65535
    assert ids.max() < 65536
    assert list(sampled_markets(32, 2)) == list(range(32))
