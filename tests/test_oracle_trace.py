"""Pins for the oracle's per-step trace and the SIV-J return statistics (SURVEY.md S8(f)-3,
DESIGN.md reading A23).  No GPU.

  * the trace is what the record says step by step (a run of S steps == S runs of one step);
  * ko_trace_stats against library routines on the same series: numpy std / mean,
    scipy.stats.kurtosis (Fisher, biased), and the textbook biased ACF estimator written with
    numpy dot products;
  * closed forms: an alternating +1/-1 return series has ACF_r(k) = (-1)^k (n-k)/n and zero
    excess-kurtosis-plus-two; a constant-|r| series has no |r| autocorrelation (0/0 -> NaN);
    a series with constant returns has zero volatility and NaN kurtosis/ACF.
"""
import numpy as np
import pytest
from scipy import stats as sps

from paper_2606_21784_b200.workloads import CONFIGS, mix3_params

REC_LAST, REC_SUMVOL = 12, 2


def _acf(x, k):
    x = np.asarray(x, dtype=np.float64)
    d = x - x.mean()
    den = float(np.dot(d, d))
    return float(np.dot(d[k:], d[:-k]) / den) if den > 0 else float("nan")


def _trace_from_prices(p, v=None):
    p = np.asarray(p, dtype=np.int32)
    t = np.zeros((len(p), 2), dtype=np.int32)
    t[:, 0] = p
    t[:, 1] = 0 if v is None else v
    return t


def test_trace_is_the_step_by_step_record(oracle):
    p = mix3_params()
    L, A, seed, ids, S = 256, 200, 4, [0, 7, 19], 40
    b, r, tr = oracle.run_markets_traced(p, L, A, seed, ids, S)
    b2, r2 = oracle.run_markets(p, L, A, seed, ids, S)
    assert np.array_equal(b, b2) and np.array_equal(r, r2)          # tracing changes nothing
    bb, rr = oracle.init_state(len(ids), L, -1)
    for t in range(S):
        vol_before = rr[:, REC_SUMVOL].copy()
        bb, rr = oracle.run_markets(p, L, A, seed, ids, 1, bb, rr)
        assert np.array_equal(tr[:, t, 0], rr[:, REC_LAST])
        assert np.array_equal(tr[:, t, 1], rr[:, REC_SUMVOL] - vol_before)
    # a traced continuation records only its own steps
    b3, r3, tr3 = oracle.run_markets_traced(p, L, A, seed, ids, 15)
    b4, r4, tr4 = oracle.run_markets_traced(p, L, A, seed, ids, 25, b3, r3)
    assert np.array_equal(np.concatenate([tr3, tr4], axis=1), tr)


@pytest.mark.parametrize("case", ["C1", "mix3", "random-walk"])
def test_trace_stats_against_numpy_and_scipy(oracle, case):
    K = 20
    if case == "C1":
        c = CONFIGS["C1"]
        _, _, tr = oracle.run_markets_traced(c.params, c.L, c.A, c.seed, [0], c.S)
        tr = tr[0]
    elif case == "mix3":
        _, _, tr = oracle.run_markets_traced(mix3_params(), 512, 300, 4, [3], 400)
        tr = tr[0]
    else:
        rng = np.random.default_rng(5)
        steps = rng.integers(-9, 10, size=3000) * (rng.random(3000) < 0.7)
        tr = _trace_from_prices(20000 + np.cumsum(steps), rng.integers(0, 500, size=3000))
    got = oracle.trace_stats(tr, K)
    r = np.diff(tr[:, 0].astype(np.int64)).astype(np.float64)
    exp = [np.std(r), sps.kurtosis(r, fisher=True, bias=True), tr[:, 1].astype(np.float64).mean(), r.mean()]
    exp += [_acf(r, k) for k in range(1, K + 1)] + [_acf(np.abs(r), k) for k in range(1, K + 1)]
    assert np.allclose(got, np.array(exp), rtol=1e-10, atol=1e-12, equal_nan=True)


def test_trace_stats_closed_forms(oracle):
    K = 4
    n = 101                                               # returns; S = n + 1 prices
    alt = 100 + (np.arange(n + 1) % 2)                    # r = +1, -1, +1, ...  (n odd: mean = 1/n)
    got = oracle.trace_stats(_trace_from_prices(alt, 7), K)
    r = np.diff(alt).astype(np.float64)
    mu = 1.0 / n
    assert got[3] == pytest.approx(mu, rel=1e-15) and got[2] == 7.0
    assert got[0] == pytest.approx(np.sqrt(1 - mu * mu), rel=1e-14)
    assert np.isnan(got[4 + K:]).all()                    # |r| is constant: 0/0
    for k in range(1, K + 1):
        # sum over t of d_t d_{t-k} with d = r - mu, r = (+1, -1, ...): evaluated exactly
        d = r - mu
        assert got[4 + k - 1] == pytest.approx(float(np.dot(d[k:], d[:-k]) / np.dot(d, d)), rel=1e-13)
        assert np.sign(got[4 + k - 1]) == (-1) ** k
    # even number of alternating returns: mean 0, ACF_r(k) = (-1)^k (n-k)/n exactly, kurtosis -2
    alt2 = 100 + (np.arange(101) % 2)
    g2 = oracle.trace_stats(_trace_from_prices(alt2), K)
    assert g2[3] == 0.0 and g2[0] == 1.0 and g2[1] == -2.0
    for k in range(1, K + 1):
        assert g2[4 + k - 1] == pytest.approx((-1) ** k * (100 - k) / 100, rel=1e-15)
    # constant drift: zero volatility, NaN kurtosis and ACFs
    g3 = oracle.trace_stats(_trace_from_prices(np.arange(50) * 3), K)
    assert g3[0] == 0.0 and g3[3] == 3.0 and np.isnan(g3[1]) and np.isnan(g3[4:]).all()
    # a single traced step: no returns at all
    g4 = oracle.trace_stats(_trace_from_prices([5], [9]), K)
    assert g4[2] == 9.0 and np.isnan(np.delete(g4, 2)).all()
