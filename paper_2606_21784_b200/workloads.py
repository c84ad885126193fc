"""Seeded, synthetic workload descriptions shared by the tests, bench.py and the oracle harness.

This module holds NONE of the method's arithmetic (no Philox, no agent rule, no clearing): it
only names the five configurations of BASELINE.json `configs`, picks which markets of a large
config are sampled for the oracle comparison, and draws random resting books for the
book-injection tests.  Both the CUDA path and the oracle are fed from here by the tests; neither
of them imports the other.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

KS_MODEL_ZI = 0
KS_MODEL_MIX3 = 1
KS_MODEL_ZI_PACKED4 = 2      # the same rules under the PACKED4 draw contract (A22)
KS_MODEL_MIX3_PACKED4 = 3


def packed4(params: dict) -> dict:
    """The same agent parameters under the PACKED4 draw contract (one Philox block per four
    consecutive agents; a separately named contract)."""
    q = dict(params)
    q["model"] = {KS_MODEL_ZI: KS_MODEL_ZI_PACKED4, KS_MODEL_MIX3: KS_MODEL_MIX3_PACKED4}[params["model"]]
    return q


KS_MODEL_PAPER = 4           # the paper's own agent model (A24)


def paper_params(A: int, alpha_mom: float, alpha_maker: float = 0.15, delta: int = 8, qmax: int = 10,
                 half_spread: int = 2, p_mkt: float = 0.05, init_price: int = -1) -> dict:
    """The paper's agent mix: class FRACTIONS turned into contiguous index
    ranges -- noise first, then round(alpha_mom*A) momentum agents, then round(alpha_maker*A)
    makers; mid-price reference, marketable orders with probability p_mkt.  The numeric values of
    delta / qmax / half_spread / p_mkt are not given in the paper: these defaults are ours."""
    n_mom, n_maker = int(round(alpha_mom * A)), int(round(alpha_maker * A))
    assert n_mom + n_maker <= A
    return dict(model=KS_MODEL_PAPER, noise_delta=delta, noise_qmax=qmax, maker_spread_max=half_spread,
                maker_qty=qmax, mom_delta=0, mom_qmax=qmax, init_price=init_price,
                paper_n_mom=n_mom, paper_n_maker=n_maker, paper_pmkt_q16=int(round(p_mkt * 65536)))


def zi_params(delta: int, qmax: int, init_price: int = -1) -> dict:
    """Zero-intelligence configs (BASELINE.json configs[0..3])."""
    return dict(model=KS_MODEL_ZI, noise_delta=delta, noise_qmax=qmax, maker_spread_max=1,
                maker_qty=1, mom_delta=0, mom_qmax=1, init_price=init_price)


def mix3_params(init_price: int = -1) -> dict:
    """Heterogeneous config (BASELINE.json configs[4]): noise [-64,64] q 1..50; maker spread 1..4
    qty 20; momentum offset [0,8] q 1..50."""
    return dict(model=KS_MODEL_MIX3, noise_delta=64, noise_qmax=50, maker_spread_max=4,
                maker_qty=20, mom_delta=8, mom_qmax=50, init_price=init_price)


@dataclass(frozen=True)
class Config:
    name: str
    M: int
    L: int
    A: int
    S: int
    seed: int
    params: dict = field(hash=False)

    @property
    def events(self) -> int:
        """agent events M*A*S (BASELINE.json `metric`)."""
        return self.M * self.A * self.S


CONFIGS = {
    "C1": Config("C1", 1, 64, 256, 100, 0, zi_params(8, 10)),
    "C2": Config("C2", 1024, 256, 1024, 1000, 1, zi_params(16, 100)),
    "C3": Config("C3", 32, 128, 512, 10000, 2, zi_params(8, 10)),
    "C4": Config("C4", 65536, 512, 4096, 1000, 3, zi_params(32, 100)),
    "C5": Config("C5", 4096, 4096, 16384, 500, 4, mix3_params()),
}


def _splitmix64_stream(state: int):
    """SplitMix64 (Steele, Lea, Flood 2014) -- used ONLY to pick which markets are sampled."""
    mask = (1 << 64) - 1
    while True:
        state = (state + 0x9E3779B97F4A7C15) & mask
        z = state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & mask
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & mask
        yield z ^ (z >> 31)


def sampled_markets(M: int, seed: int, n: int = 64) -> np.ndarray:
    """Market ids the oracle is run on for a large config: {0, M-1} plus the first n-2 distinct
    values of floor(hi32(SplitMix64) * M / 2^32), stream seeded with 0xC0FFEE ^ seed.  If M <= n,
    every market."""
    if M <= n:
        return np.arange(M, dtype=np.uint32)
    ids = [0, M - 1]
    seen = set(ids)
    for z in _splitmix64_stream(0xC0FFEE ^ seed):
        v = ((z >> 32) * M) >> 32
        if v not in seen:
            seen.add(v)
            ids.append(v)
            if len(ids) == n:
                break
    return np.array(ids, dtype=np.uint32)


def random_books(n: int, L: int, seed: int, max_qty: int = 50, fill: float = 0.5,
                 crossed: bool = True) -> np.ndarray:
    """Random resting books int32 [n][2][L] for the book-injection tests (numpy PCG64 stream).

    `fill` is the probability that a (side, tick) cell is non-empty.  With crossed=False the
    bids are confined to the lower half and the asks to the upper half of the grid.
    """
    rng = np.random.default_rng(seed)
    q = rng.integers(1, max_qty + 1, size=(n, 2, L), dtype=np.int64)
    mask = rng.random(size=(n, 2, L)) < fill
    books = (q * mask).astype(np.int32)
    if not crossed:
        books[:, 0, L // 2:] = 0
        books[:, 1, :L // 2] = 0
    return books


def shard_markets(M: int, rank: int, world: int):
    """Contiguous partition of the market range [0, M) across `world` ranks -> (base, count).
    Markets are independent, so this is the whole multi-GPU story."""
    q, r = divmod(M, world)
    base = rank * q + min(rank, r)
    return base, q + (1 if rank < r else 0)
