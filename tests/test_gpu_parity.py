"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle on
the same seeded configurations -- bit-exact on books, clearing prices (trajectory hash), every
integer sum; derived fp64 statistics within 1e-12 relative (north_star)."""
import numpy as np
import pytest

from ks_testlib import assert_rows_equal, ints, oracle_rows, read_golden
from paper_2606_21784_b200.workloads import (CONFIGS, mix3_params, packed4, paper_params, random_books,
                                             sampled_markets, zi_params)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ks():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2606_21784_b200 import binding
    binding.load()          # raises if the CUDA library is not built: no fallback
    return binding


def _gpu(ks, M, L, A, params, seed, S, *, opts=(), market_base=0, books=None, split=None, stepwise=False):
    import torch
    sim = ks.KsSim(M, L, A, params, seed, market_base=market_base)
    for o, v in opts:
        sim.ks_set_option(o, v)
    if books is not None:
        sim.ks_write_books(torch.from_numpy(np.ascontiguousarray(books)).cuda())
    for s in (split or [S]):
        (sim.ks_run_stepwise if stepwise else sim.ks_run)(s)
    b, r = sim.books_to_host(), sim.stats_to_host()
    sim.ks_destroy()
    return b, r


def _check_derived(ks, oracle, recs):
    got = ks.ks_derive_stats(recs)
    exp = np.stack([oracle.derived(r) for r in recs])
    assert np.array_equal(np.isnan(got), np.isnan(exp))
    m = ~np.isnan(exp)
    assert np.all(np.abs(got[m] - exp[m]) <= 1e-12 * np.abs(exp[m]))


# ------------------------------------------------------------------ the five BASELINE configs
@pytest.mark.parametrize("name", ["C1", "C2", "C3"])
def test_config_all_markets(ks, oracle, name):
    """C1-C3 at full size, every market (C2 is ~1e9 agent events for the oracle)."""
    c = CONFIGS[name]
    b, r = _gpu(ks, c.M, c.L, c.A, c.params, c.seed, c.S)
    ids = np.arange(c.M)
    eb, er = oracle_rows(oracle, c.params, c.L, c.A, c.seed, ids, c.S)
    assert_rows_equal(b, r, ids, eb, er, name)
    _check_derived(ks, oracle, r)


@pytest.mark.parametrize("name", ["C4", "C5"])
def test_config_sampled_markets(ks, oracle, name):
    """C4/C5 at BASELINE.json's full size in the launch configuration bench.py times; the oracle
    runs the 64 seeded sampled markets (ids 0, M-1 and 62 SplitMix64 draws)."""
    c = CONFIGS[name]
    b, r = _gpu(ks, c.M, c.L, c.A, c.params, c.seed, c.S)
    ids = sampled_markets(c.M, c.seed, 64)
    eb, er = oracle_rows(oracle, c.params, c.L, c.A, c.seed, ids, c.S)
    assert_rows_equal(b, r, ids, eb, er, name)
    _check_derived(ks, oracle, r[ids.astype(np.int64)])
    # properties that hold for every market at any size
    r64 = r.astype(np.int64)
    assert (r64[:, 0] == c.S).all() and (r64[:, 1] <= c.S).all()
    assert (b >= 0).all()
    tot = b.astype(np.int64).sum(axis=2)
    assert (r64[:, 10] == r64[:, 2] + tot[:, 0]).all() and (r64[:, 11] == r64[:, 2] + tot[:, 1]).all()


# ------------------------------------------------------------------ equivalences
@pytest.mark.parametrize("model", ["zi", "mix3"])
def test_block_sizes_atomic_modes_and_clear_paths_give_identical_bytes(ks, oracle, model):
    """Integer quantities make accumulation order irrelevant: any block size, the
    warp-aggregated atomics and the chunked general scan must give the same bytes as the oracle.
    Ragged sizes: A is not a multiple of the block size or of 3."""
    if model == "zi":
        M, L, A, S, seed, p = 37, 256, 1000, 120, 9, zi_params(16, 100)
    else:
        M, L, A, S, seed, p = 21, 1024, 1541, 90, 4, mix3_params()
    ids = np.arange(M)
    eb, er = oracle_rows(oracle, p, L, A, seed, ids, S)
    for T in (32, 64, 96, 128, 256, 512, 1024):
        for atom in (0, 1):
            for clear in (0, 1):
                if T not in (32, 96, 256, 1024) and (atom or clear):
                    continue
                b, r = _gpu(ks, M, L, A, p, seed, S, opts=[(ks.KS_OPT_BLOCK_THREADS, T),
                                                            (ks.KS_OPT_ATOMIC_MODE, atom),
                                                            (ks.KS_OPT_CLEAR_PATH, clear)])
                assert_rows_equal(b, r, ids, eb, er, "T=%d atom=%d clear=%d" % (T, atom, clear))


def test_decoupled_kernel_gives_identical_bytes(ks, oracle):
    """KS_OPT_PIPELINE: ks_decoupled_kernel -- generating warps fill a price-independent relative
    order histogram (a ring of 4, or 2, histograms: up to that many steps ahead), one clearing warp per market merges
    it at the step's price.  Forced on (2) and off (1) for several block sizes and ragged agent
    counts, plain bins and the 32-lane-column layout, literal and PACKED4 draws, prices pinned to the
    grid edges (the clamp happens at the merge), split and launch-per-step runs, S = 1 .. 5 (the
    ring's corner cases), the trace: always the oracle's bytes."""
    import torch
    L, seed, S = 128, 2, 150
    p = zi_params(8, 10)
    # (pipe = 1, ks_persistent_kernel: clearing warp = market mod #warps, so M > #warps makes every warp index a
    # clearing warp; ks_decoupled_kernel's clearing warp is always the CTA's last warp)
    for M, A, T in [(5, 512, 512), (5, 500, 256), (3, 97, 64), (4, 33, 96), (2, 0, 128), (3, 1900, 512), (2, 1984, 1024),
                    (7, 1024, 160), (6, 1024, 128), (9, 1000, 96), (5, 3000, 224), (11, 4096, 1024), (3, 4096, 288)]:
        ids = np.arange(M)
        eb, er = oracle_rows(oracle, p, L, A, seed, ids, S)
        for pipe, cols, ring in ((2, 0, 0), (2, 0, 2), (2, 1, 0), (1, 0, 0)):
            b, r = _gpu(ks, M, L, A, p, seed, S, opts=[(ks.KS_OPT_BLOCK_THREADS, T), (ks.KS_OPT_PIPELINE, pipe),
                                                        (ks.KS_OPT_REL_COLUMNS, cols), (ks.KS_OPT_RING_DEPTH, ring)])
            assert_rows_equal(b, r, ids, eb, er, "decoupled=%d cols=%d ring=%d A=%d T=%d" % (pipe, cols, ring, A, T))
    # the C2 shape's window (delta = 16: 33 ticks, the two-row fused scan), 7 markets of 160 threads
    p2 = zi_params(16, 100)
    for M, A, T in [(9, 1024, 160), (5, 777, 128), (3, 2000, 544)]:
        eb, er = oracle_rows(oracle, p2, 256, A, 1, np.arange(M), 90)
        for ring in (0, 2):
            b, r = _gpu(ks, M, 256, A, p2, 1, 90, opts=[(ks.KS_OPT_BLOCK_THREADS, T), (ks.KS_OPT_PIPELINE, 2),
                                                        (ks.KS_OPT_RING_DEPTH, ring)])
            assert_rows_equal(b, r, np.arange(M), eb, er, "decoupled C2 shape ring=%d A=%d T=%d" % (ring, A, T))
    pk = packed4(zi_params(16, 100))
    for M, A, T in [(6, 1001, 128), (5, 3, 64), (7, 4096, 288)]:
        eb, er = oracle_rows(oracle, pk, 256, A, 9, np.arange(M), 70)
        for cols in (0, 1):
            b, r = _gpu(ks, M, 256, A, pk, 9, 70, opts=[(ks.KS_OPT_BLOCK_THREADS, T), (ks.KS_OPT_PIPELINE, 2),
                                                        (ks.KS_OPT_REL_COLUMNS, cols)])
            assert_rows_equal(b, r, np.arange(M), eb, er, "decoupled packed4 cols=%d A=%d T=%d" % (cols, A, T))
    M, A, T = 4, 480, 256
    ids = np.arange(M)
    for init in (0, L - 1, 4):
        q = dict(p, init_price=init)
        eb, er, et = oracle.run_markets_traced(q, L, A, seed, ids, 60)
        for kw in (dict(), dict(split=[1, 29, 30]), dict(split=[2, 3, 55]), dict(split=[4, 5, 51]), dict(stepwise=True)):
            for cols in (0, 1):
                b, r = _gpu(ks, M, L, A, q, seed, 60, opts=[(ks.KS_OPT_BLOCK_THREADS, T), (ks.KS_OPT_PIPELINE, 2),
                                                            (ks.KS_OPT_REL_COLUMNS, cols)], **kw)
                assert_rows_equal(b, r, ids, eb, er, "decoupled init=%d cols=%d %r" % (init, cols, kw))
        sim = ks.KsSim(M, L, A, q, seed)
        sim.ks_set_option(ks.KS_OPT_BLOCK_THREADS, T); sim.ks_set_option(ks.KS_OPT_PIPELINE, 2)
        tr = torch.empty((M, 60, 2), dtype=torch.int32, device="cuda")
        sim.ks_run_traced(60, tr)
        assert np.array_equal(tr.cpu().numpy(), et)
        sim.ks_destroy()
    # injected crossed books + a wide offset range (2 x 257 bins, several merge rounds)
    M, L2, A = 5, 1024, 700
    pw = zi_params(128, 30)
    books = random_books(M, L2, seed=11, max_qty=40, fill=0.2)
    eb0, er0 = oracle.init_state(M, L2, -1)
    eb, er = oracle_rows(oracle, pw, L2, A, 3, np.arange(M), 25, books=books, recs=er0)
    for cols in (0, 1):
        b, r = _gpu(ks, M, L2, A, pw, 3, 25, books=books, opts=[(ks.KS_OPT_BLOCK_THREADS, 192), (ks.KS_OPT_PIPELINE, 2),
                                                                (ks.KS_OPT_REL_COLUMNS, cols)])
        assert_rows_equal(b, r, np.arange(M), eb, er, "decoupled injected cols=%d" % cols)


@pytest.mark.parametrize("group", [2])
def test_step_pairs_give_identical_bytes(ks, oracle, group):
    """KS_OPT_STEP_PAIRS: the decoupled kernel's generating warps make two steps per pass
    over their agents (shared step-independent Philox rounds) and hand them over together; the
    clearing warp keeps the record.  Step counts that leave a partial last group, split and
    launch-per-step runs (a group never spans two ks_run calls), ragged agent counts, grid-edge
    prices (clamped at the merge), the trace, the C2 and C4 shapes' windows: the oracle's bytes."""
    import torch
    opts = [(ks.KS_OPT_PIPELINE, 2), (ks.KS_OPT_STEP_PAIRS, group)]
    for (M, L, A, delta, qmax, T, S) in [(9, 256, 1024, 16, 100, 160, 91), (5, 512, 4096, 32, 100, 160, 40), (7, 128, 300, 8, 10, 160, 75),
                                         (3, 256, 1000, 16, 100, 96, 33), (4, 128, 33, 8, 10, 64, 50), (2, 64, 0, 8, 10, 160, 9)]:
        p = zi_params(delta, qmax)
        ids = np.arange(M)
        eb, er = oracle_rows(oracle, p, L, A, 3, ids, S)
        for kw in (dict(), dict(split=[1, 2, S - 3]), dict(split=[3, S - 8, 5]), dict(stepwise=True)):
            b, r = _gpu(ks, M, L, A, p, 3, S, opts=opts + [(ks.KS_OPT_BLOCK_THREADS, T)], **kw)
            assert_rows_equal(b, r, ids, eb, er, "pairs M=%d A=%d T=%d S=%d %r" % (M, A, T, S, kw))
    for S in (1, 2, 3, 4, 5, 6, 7, 8, 9, 11, 13):
        p = zi_params(16, 100)
        eb, er = oracle_rows(oracle, p, 256, 700, 8, np.arange(4), S)
        b, r = _gpu(ks, 4, 256, 700, p, 8, S, opts=opts + [(ks.KS_OPT_BLOCK_THREADS, 160)])
        assert_rows_equal(b, r, np.arange(4), eb, er, "pairs S=%d" % S)
    M, L, A = 4, 128, 480
    for init in (0, L - 1, 5):
        q = dict(zi_params(8, 10), init_price=init)
        eb, er, et = oracle.run_markets_traced(q, L, A, 2, np.arange(M), 61)
        sim = ks.KsSim(M, L, A, q, 2)
        for o, v in opts + [(ks.KS_OPT_BLOCK_THREADS, 160)]:
            sim.ks_set_option(o, v)
        tr = torch.empty((M, 61, 2), dtype=torch.int32, device="cuda")
        sim.ks_run_traced(61, tr)
        b, r = sim.books_to_host(), sim.stats_to_host()
        sim.ks_destroy()
        assert_rows_equal(b, r, np.arange(M), eb, er, "pairs traced init=%d" % init)
        assert np.array_equal(tr.cpu().numpy(), et)


def test_mix3_decoupled_gives_identical_bytes(ks, oracle):
    """The three-type population under the decoupled kernel (two steps per pass): noise, maker and
    momentum orders go into histograms relative to the step's opening price -- makers one bin per
    spread (added to both sides at the merge), momentum one bin per offset plus the coin-says-buy
    share that decides a flat price -- and the clearing warp merges them at the step's price and
    price change.  Forced on for several shapes, ragged agent counts (every class gets a tail),
    odd and tiny step counts, split / launch-per-step runs, prices pinned to both grid edges (clamps
    at the merge), flat-price starts (the coin path), other parameter values, the trace."""
    import torch
    opts = [(ks.KS_OPT_PIPELINE, 2)]
    for (M, L, A, T, S, p) in [(7, 1024, 1541, 160, 45, mix3_params()), (5, 4096, 6000, 160, 31, mix3_params()),
                               (4, 256, 100, 96, 60, mix3_params()), (3, 512, 7, 64, 20, mix3_params()),
                               (6, 128, 900, 128, 50, dict(mix3_params(), noise_delta=20, maker_spread_max=9, mom_delta=30,
                                                           noise_qmax=7, mom_qmax=3, maker_qty=1))]:
        ids = np.arange(M)
        eb, er = oracle_rows(oracle, p, L, A, 4, ids, S)
        for kw in (dict(), dict(split=[1, 2, S - 3]), dict(split=[3, S - 8, 5]), dict(stepwise=True)):
            b, r = _gpu(ks, M, L, A, p, 4, S, opts=opts + [(ks.KS_OPT_BLOCK_THREADS, T)], **kw)
            assert_rows_equal(b, r, ids, eb, er, "mix3 decoupled M=%d L=%d A=%d T=%d %r" % (M, L, A, T, kw))
    for S in (1, 2, 3, 4, 5, 7):
        eb, er = oracle_rows(oracle, mix3_params(), 512, 700, 8, np.arange(4), S)
        b, r = _gpu(ks, 4, 512, 700, mix3_params(), 8, S, opts=opts + [(ks.KS_OPT_BLOCK_THREADS, 160)])
        assert_rows_equal(b, r, np.arange(4), eb, er, "mix3 decoupled S=%d" % S)
    M, L, A = 4, 256, 600
    for init in (0, L - 1, 3, L - 5):
        q = dict(mix3_params(), init_price=init)
        eb, er, et = oracle.run_markets_traced(q, L, A, 2, np.arange(M), 41)
        sim = ks.KsSim(M, L, A, q, 2)
        for o, v in opts + [(ks.KS_OPT_BLOCK_THREADS, 160)]:
            sim.ks_set_option(o, v)
        assert "mix3" in sim.ks_plan_string()
        tr = torch.empty((M, 41, 2), dtype=torch.int32, device="cuda")
        sim.ks_run_traced(41, tr)
        b, r = sim.books_to_host(), sim.stats_to_host()
        sim.ks_destroy()
        assert_rows_equal(b, r, np.arange(M), eb, er, "mix3 decoupled traced init=%d" % init)
        assert np.array_equal(tr.cpu().numpy(), et)
    # injected crossed books (wide first window) and checkpoint attach
    books = random_books(3, 512, seed=5, max_qty=30, fill=0.1)
    eb0, er0 = oracle.init_state(3, 512, -1)
    eb, er = oracle_rows(oracle, mix3_params(), 512, 800, 6, np.arange(3), 25, books=books, recs=er0)
    b, r = _gpu(ks, 3, 512, 800, mix3_params(), 6, 25, books=books, opts=opts + [(ks.KS_OPT_BLOCK_THREADS, 160)])
    assert_rows_equal(b, r, np.arange(3), eb, er, "mix3 decoupled injected")


def test_split_run_and_stepwise_ablation_are_bit_identical(ks, oracle):
    """ks_run(S1); ks_run(S2) == ks_run(S1+S2); the launch-per-step ablation (a8) == persistent."""
    c = CONFIGS["C3"]
    S = 300
    ids = np.arange(c.M)
    eb, er = oracle_rows(oracle, c.params, c.L, c.A, c.seed, ids, S)
    b1, r1 = _gpu(ks, c.M, c.L, c.A, c.params, c.seed, S)
    b2, r2 = _gpu(ks, c.M, c.L, c.A, c.params, c.seed, S, split=[1, 99, 200])
    b3, r3 = _gpu(ks, c.M, c.L, c.A, c.params, c.seed, S, stepwise=True)
    for b, r, what in [(b1, r1, "one run"), (b2, r2, "split"), (b3, r3, "stepwise")]:
        assert_rows_equal(b, r, ids, eb, er, what)
    m = mix3_params()
    eb, er = oracle_rows(oracle, m, 512, 700, 4, np.arange(5), 64)
    b, r = _gpu(ks, 5, 512, 700, m, 4, 64, split=[7, 57])
    assert_rows_equal(b, r, np.arange(5), eb, er, "mix3 split")
    b, r = _gpu(ks, 5, 512, 700, m, 4, 64, stepwise=True)
    assert_rows_equal(b, r, np.arange(5), eb, er, "mix3 stepwise")


def test_market_base_shards_reproduce_the_global_run(ks, oracle):
    """S8(e): a shard created with market_base = b computes markets b..b+M-1 of the global run."""
    c = CONFIGS["C2"]
    S = 40
    bg, rg = _gpu(ks, 64, c.L, c.A, c.params, c.seed, S)
    b0, r0 = _gpu(ks, 24, c.L, c.A, c.params, c.seed, S)
    b1, r1 = _gpu(ks, 40, c.L, c.A, c.params, c.seed, S, market_base=24)
    assert np.array_equal(np.concatenate([b0, b1]), bg) and np.array_equal(np.concatenate([r0, r1]), rg)
    eb, er = oracle_rows(oracle, c.params, c.L, c.A, c.seed, np.arange(24, 64), S)
    assert_rows_equal(b1, r1, np.arange(40), eb, er, "shard with market_base")


# ------------------------------------------------------------------ cluster / DSMEM path
@pytest.mark.parametrize("model", ["zi", "mix3"])
def test_cluster_path_gives_identical_bytes(ks, oracle, model):
    """north_star (2): the book split across the CTAs of a thread-block cluster (remote
    shared-memory reductions, clearing through ld/st.shared::cluster) must give the bytes of the
    oracle for every cluster size, block size, clearing path, split run and injected book."""
    if model == "zi":
        M, L, A, S, seed, p = 19, 256, 1000, 80, 9, zi_params(16, 100)
    else:
        M, L, A, S, seed, p = 11, 1024, 1541, 60, 4, mix3_params()
    ids = np.arange(M)
    eb, er = oracle_rows(oracle, p, L, A, seed, ids, S)
    for C in (2, 4, 8):
        for T, clear, split in ((0, 0, None), (32, 1, None), (96, 0, [1, S - 1]), (1024, 0, None)):
            b, r = _gpu(ks, M, L, A, p, seed, S, split=split,
                        opts=[(ks.KS_OPT_CLUSTER_SIZE, C), (ks.KS_OPT_BLOCK_THREADS, T), (ks.KS_OPT_CLEAR_PATH, clear)])
            assert_rows_equal(b, r, ids, eb, er, "cluster C=%d T=%d clear=%d" % (C, T, clear))
    # injected crossed books that span every CTA of the cluster; price pinned near a CTA boundary
    books = random_books(M, L, seed=77, max_qty=40, fill=0.3)
    eb0, er0 = oracle.init_state(M, L, -1)
    eb, er = oracle_rows(oracle, p, L, A, seed, ids, 7, books=books, recs=er0)
    for C in (2, 8):
        b, r = _gpu(ks, M, L, A, p, seed, 7, books=books, opts=[(ks.KS_OPT_CLUSTER_SIZE, C)])
        assert_rows_equal(b, r, ids, eb, er, "cluster injected C=%d" % C)


def test_book_larger_than_one_sm(ks, oracle):
    """L = 32768: 256 KB of book per market, more than one SM's shared memory -> the automatic
    plan runs a 2-CTA cluster.  Opening price at the CTA boundary (L/2), so orders and the
    clearing window straddle both CTAs' shared memory.  S = 1000 steps: the a-priori
    (L-1)^4 * steps < 2^63 guard of round 1 (8 steps at this L) is gone -- the int64 sums are
    checked exactly on the device, and these runs stay far inside them."""
    M, L, A, S, seed = 4, 32768, 300, 1000, 21
    p = zi_params(64, 50)
    ids = np.arange(M)
    eb, er = oracle_rows(oracle, p, L, A, seed, ids, S)
    b, r = _gpu(ks, M, L, A, p, seed, S, split=[400, 600])
    assert_rows_equal(b, r, ids, eb, er, "L=32768 auto cluster, S=1000")
    pm = mix3_params()
    books = random_books(M, L, seed=5, max_qty=30, fill=0.05)
    eb0, er0 = oracle.init_state(M, L, -1)
    eb, er = oracle_rows(oracle, pm, L, 900, seed, ids, 40, books=books, recs=er0)
    b, r = _gpu(ks, M, L, 900, pm, seed, 40, books=books, split=[2, 38])
    assert_rows_equal(b, r, ids, eb, er, "L=32768 mix3 injected")


def test_large_price_moves_reach_the_int64_limit_exactly(ks, oracle):
    """The sum of r^4 (f[9]) is the statistic that can leave int64 on a wide grid.  A = 0 and
    injected crossed quotes (ks_write_books before every step) make the price jump between tick 10
    and tick 32700 of an L = 32768 grid: the first jump from L/2 adds 16374^4, each later one
    32690^4 = 1.142e18.  After 1 + 8 jumps the sum is 9.208e18 < 2^63 = 9.223e18 and every byte
    still equals the oracle's (whose int64 sums have not overflowed either); the next jump leaves
    int64, the kernel raises the sticky flag and the handle returns KS_ERR_OVERFLOW from then on."""
    import torch
    M, L, seed, p = 3, 32768, 1, zi_params(8, 10)
    ids = np.arange(M)

    def quotes(k):
        b = np.zeros((M, 2, L), dtype=np.int32)
        lo, hi = (10, 32700) if k % 2 == 0 else (32700, 32750)     # ask at lo, bid at hi: V = q on [lo, hi], p* = lo
        b[:, 1, lo] = 5 + np.arange(M); b[:, 0, hi] = 5 + np.arange(M)
        return b

    sim = ks.KsSim(M, L, 0, p, seed)
    eb, er = oracle.init_state(M, L, -1)
    for k in range(9):
        sim.ks_write_books(torch.from_numpy(quotes(k)).cuda())
        sim.ks_run(1)
        eb, er = oracle.run_markets(p, L, 0, seed, ids.astype(np.uint32), 1, quotes(k), er)
    torch.cuda.synchronize()
    sim.ks_error_state()
    assert_rows_equal(sim.books_to_host(), sim.stats_to_host(), ids, eb, er, "nine jumps")
    assert (er[:, 12] == 10).all() and (er[:, 9] == 16374 ** 4 + 8 * 32690 ** 4).all() and (er[:, 9] > 0.998 * 2 ** 63).all()
    sim.ks_write_books(torch.from_numpy(quotes(9)).cuda())
    sim.ks_run(1)
    torch.cuda.synchronize()
    for call in (sim.ks_error_state, lambda: sim.ks_run(1), sim.stats_to_host):
        with pytest.raises(ks.KsError) as e:
            call()
        assert e.value.status == ks.KS_ERR_OVERFLOW
    sim.ks_destroy()


def test_single_cta_maximum_grid_long_run(ks, oracle):
    """L = 16384 (the single-CTA maximum), S = 1000 (round 1's guard allowed 128 steps)."""
    M, L, A, S, seed = 3, 16384, 400, 1000, 8
    p = zi_params(100, 20)
    eb, er = oracle_rows(oracle, p, L, A, seed, np.arange(M), S)
    b, r = _gpu(ks, M, L, A, p, seed, S)
    assert_rows_equal(b, r, np.arange(M), eb, er, "L=16384, S=1000")


# ------------------------------------------------------------------ checkpoint / deferred errors
@pytest.mark.parametrize("case", ["zi", "mix3", "paper", "cluster", "decoupled"])
def test_checkpoint_attach_resumes_bit_exactly(ks, oracle, case):
    """include/kineticsim.h: d_state IS the checkpoint.  Save its bytes after S1 steps, destroy the
    handle, scribble over the buffer, restore the bytes, ks_attach a NEW handle, run S2 more steps:
    the result equals one uninterrupted run of S1 + S2 steps (and the oracle)."""
    import torch
    opts = []
    if case == "zi":
        M, L, A, seed, p = 11, 256, 700, 9, zi_params(16, 100)
    elif case == "mix3":
        M, L, A, seed, p = 7, 1024, 900, 4, mix3_params()
    elif case == "paper":
        M, L, A, seed, p = 9, 128, 200, 5, paper_params(200, 0.15, 0.15, p_mkt=0.05)
    elif case == "cluster":
        M, L, A, seed, p = 5, 512, 600, 8, zi_params(32, 50)
        opts = [(ks.KS_OPT_CLUSTER_SIZE, 4)]
    else:
        M, L, A, seed, p = 6, 128, 512, 2, zi_params(8, 10)
        opts = [(ks.KS_OPT_BLOCK_THREADS, 256), (ks.KS_OPT_PIPELINE, 2)]      # ks_decoupled_kernel
    S1, S2 = 37, 55
    ids = np.arange(M)
    eb, er = oracle_rows(oracle, p, L, A, seed, ids, S1 + S2)
    sim = ks.KsSim(M, L, A, p, seed)
    for o, v in opts:
        sim.ks_set_option(o, v)
    sim.ks_run(S1)
    torch.cuda.synchronize()
    saved = sim.state.clone()
    sim.ks_destroy()
    state = torch.full_like(saved, 0x5A)                # a different buffer with garbage in it
    state.copy_(saved)
    sim2 = ks.KsSim(M, L, A, p, seed, state=state, attach=True)
    for o, v in opts:
        sim2.ks_set_option(o, v)
    sim2.ks_run(S2)
    b, r = sim2.books_to_host(), sim2.stats_to_host()
    sim2.ks_destroy()
    assert_rows_equal(b, r, ids, eb, er, "attach " + case)
    # the guards of the new handle start from the restored step counter and depth, not from zero
    sim3 = ks.KsSim(M, L, A, p, seed, state=state, attach=True)
    with pytest.raises(ks.KsError) as e:
        sim3.ks_run(2 ** 32 - (S1 + S2))
    assert e.value.status == ks.KS_ERR_OVERFLOW
    sim3.ks_destroy()


def test_statistic_overflow_is_detected_on_the_device(ks):
    """The int64 sum of r^4 (f[9]) is checked exactly where it is formed: a record restored with
    f[9] just below 2^63 overflows at the first price move, the kernel raises the sticky flag, and
    every later call on the handle returns KS_ERR_OVERFLOW.  The same state with f[9] = 0 runs."""
    import torch
    M, L, A, seed, p = 3, 64, 256, 0, zi_params(8, 10)
    sim = ks.KsSim(M, L, A, p, seed)
    sim.ks_run(5)
    torch.cuda.synchronize()
    state = sim.state.clone()
    sim.ks_destroy()
    recs = state[M * 8 * L: M * (8 * L + 128)].view(torch.int64).view(M, 16)
    ok = ks.KsSim(M, L, A, p, seed, state=state.clone(), attach=True)
    ok.ks_run(200); torch.cuda.synchronize(); ok.ks_error_state()
    moved = ok.stats_to_host()[:, 7] > 0                      # sum r^2 > 0: the price moved
    ok.ks_destroy()
    assert moved[1]
    recs[1, 9] = 2 ** 63 - 1                                   # market 1 only
    bad = ks.KsSim(M, L, A, p, seed, state=state, attach=True)
    bad.ks_error_state()
    bad.ks_run(200)
    torch.cuda.synchronize()
    for call in (bad.ks_error_state, lambda: bad.ks_run(1), bad.stats_to_host, bad.books_to_host):
        with pytest.raises(ks.KsError) as e:
            call()
        assert e.value.status == ks.KS_ERR_OVERFLOW
    bad.ks_destroy()


def test_deferred_depth_check_refuses_the_run_on_the_device(ks, oracle):
    """ks_run right after ks_write_books does not wait for the depth check: when the injected depth
    plus the run's inflow could reach 2^31 the kernel itself refuses, nothing changes, and the
    error surfaces as a sticky KS_ERR_OVERFLOW; a negative depth gives KS_ERR_INVALID_ARG.  A legal
    injected book runs exactly as before (every other injected-book test takes this path too)."""
    import torch
    M, L, A, seed, p = 4, 64, 100, 3, zi_params(8, 10)
    for poison, status in ((2 ** 31 - 1000, ks.KS_ERR_OVERFLOW), (-1, ks.KS_ERR_INVALID_ARG)):
        books = random_books(M, L, seed=1, max_qty=20, fill=0.3)
        books[2, 1, 7] = poison
        d_books = torch.from_numpy(books).cuda()
        sim = ks.KsSim(M, L, A, p, seed)
        sim.ks_write_books(d_books)
        try:
            sim.ks_run(10)                                 # usually enqueued: the check is still in flight
            torch.cuda.synchronize()
            with pytest.raises(ks.KsError) as e:
                sim.ks_error_state()
            assert e.value.status == status
        except ks.KsError as e2:                           # the host already had the result
            assert e2.status == status
        torch.cuda.synchronize()
        raw = sim.state[: M * 8 * L].view(torch.int32).view(M, 2, L).cpu().numpy()
        rec = sim.state[M * 8 * L: M * (8 * L + 128)].view(torch.int64).view(M, 16).cpu().numpy()
        assert np.array_equal(raw, books) and (rec[:, 0] == 0).all()     # not a byte of the run happened
        sim.ks_destroy()


def test_attach_checks_every_markets_record(ks):
    """ks_attach adopts per-market step counters and prices: a record that this library cannot have
    written -- in ANY market, not only market 0 -- is refused (a price off the grid would reach the
    rules' tick arithmetic unclamped), and the run guards continue from the largest step counter."""
    import torch
    M, L, A, seed, p = 6, 64, 100, 3, zi_params(8, 10)
    sim = ks.KsSim(M, L, A, p, seed)
    sim.ks_run(20)
    torch.cuda.synchronize()
    good = sim.state.clone()
    sim.ks_destroy()
    rec0 = M * 8 * L
    for m, field, value in ((4, 12, L), (5, 12, -1), (3, 13, L + 5), (2, 13, -2), (1, 0, -7)):
        state = good.clone()
        state[rec0: rec0 + M * 128].view(torch.int64).view(M, 16)[m, field] = value
        with pytest.raises(ks.KsError) as e:
            ks.KsSim(M, L, A, p, seed, state=state, attach=True)
        assert e.value.status == ks.KS_ERR_INVALID_ARG, (m, field, value)
    # a market further along than market 0: the step guard counts from the maximum
    state = good.clone()
    state[rec0: rec0 + M * 128].view(torch.int64).view(M, 16)[4, 0] = 2 ** 32 - 100
    sim = ks.KsSim(M, L, A, p, seed, state=state, attach=True)
    with pytest.raises(ks.KsError) as e:
        sim.ks_run(95)
    assert e.value.status == ks.KS_ERR_OVERFLOW
    sim.ks_destroy()
    # KS_MODEL_PAPER keeps the doubled mid in f[13]: up to 2(L-1) is legal there
    pp = paper_params(100, 0.15, 0.15)
    sim = ks.KsSim(M, L, 100, pp, seed)
    sim.ks_run(5)
    torch.cuda.synchronize()
    state = sim.state.clone()
    sim.ks_destroy()
    state[rec0: rec0 + M * 128].view(torch.int64).view(M, 16)[2, 13] = 2 * (L - 1)
    ks.KsSim(M, L, 100, pp, seed, state=state, attach=True).ks_destroy()
    state[rec0: rec0 + M * 128].view(torch.int64).view(M, 16)[2, 13] = 2 * L - 1
    with pytest.raises(ks.KsError):
        ks.KsSim(M, L, 100, pp, seed, state=state, attach=True)


def test_step_counter_guard_leaves_headroom_for_the_kernels_lookahead(ks):
    """The kernels count steps in 32 bits and the decoupled kernel compares `s + stride < S` with a
    stride of up to 8: ks_run refuses a run that would bring the counter within 8 of 2^32."""
    M, L, A, seed, p = 2, 64, 0, 1, zi_params(8, 10)
    sim = ks.KsSim(M, L, A, p, seed)
    for S in (2 ** 32 - 8, 2 ** 32 - 1, 2 ** 32):
        with pytest.raises(ks.KsError) as e:
            sim.ks_run(S)
        assert e.value.status == ks.KS_ERR_OVERFLOW
    sim.ks_destroy()


def test_run_on_another_stream_than_write_books(ks, oracle):
    """ks_run reads the pending depth check's word on the device; the library orders the launch after
    the check with an event wait, so the run may be enqueued on a different stream than
    ks_write_books (the books themselves are the caller's to order: done here with an event)."""
    import torch
    M, L, A, seed, S, p = 40, 256, 300, 6, 25, zi_params(16, 50)
    books = random_books(M, L, seed=9, max_qty=30, fill=0.4)
    _, er0 = oracle.init_state(M, L, -1)
    eb, er = oracle_rows(oracle, p, L, A, seed, np.arange(M), S, books=books, recs=er0)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    d_books = torch.from_numpy(books).cuda()
    torch.cuda.synchronize()
    sim = ks.KsSim(M, L, A, p, seed, stream=s1)
    filler = torch.empty(1 << 28, dtype=torch.uint8, device="cuda")
    with torch.cuda.stream(s1):
        for _ in range(8):
            filler.fill_(1)                             # keeps s1 busy so that the check is still pending
    sim.ks_write_books(d_books, stream=s1)
    ev = torch.cuda.Event()
    ev.record(s1)
    s2.wait_event(ev)
    sim.ks_run(S, stream=s2)
    s2.synchronize()
    b, r = sim.books_to_host(), sim.stats_to_host()
    sim.ks_destroy()
    assert_rows_equal(b, r, np.arange(M), eb, er, "run on another stream")


# ------------------------------------------------------------------ PACKED4 draw contract
@pytest.mark.parametrize("model", ["zi", "mix3"])
def test_packed4_contract_matches_the_oracle(ks, oracle, model):
    """SURVEY.md S8(f)-1 / DESIGN.md A22: one Philox block per four agents, draws by successive
    multiply-extract.  Ragged agent counts (A mod 4 = 0..3, A < 4), every block size, both
    clearing paths, split and launch-per-step runs, the cluster path, prices pinned to the grid
    edges (clamp path) -- all bit-exact against the oracle's PACKED4 mode."""
    if model == "zi":
        M, L, S, seed, p = 23, 256, 70, 9, packed4(zi_params(16, 100))
    else:
        M, L, S, seed, p = 13, 1024, 50, 4, packed4(mix3_params())
    ids = np.arange(M)
    for A in (1000, 1001, 1002, 1003, 3, 0):
        eb, er = oracle_rows(oracle, p, L, A, seed, ids, S)
        for T in ((0, 32, 96, 1024) if A == 1001 else (0,)):
            b, r = _gpu(ks, M, L, A, p, seed, S, opts=[(ks.KS_OPT_BLOCK_THREADS, T)])
            assert_rows_equal(b, r, ids, eb, er, "packed4 A=%d T=%d" % (A, T))
    A = 1001
    eb, er = oracle_rows(oracle, p, L, A, seed, ids, S)
    for kw in (dict(split=[1, 9, S - 10]), dict(stepwise=True), dict(opts=[(ks.KS_OPT_CLEAR_PATH, 1)]),
               dict(opts=[(ks.KS_OPT_CLUSTER_SIZE, 2)]), dict(opts=[(ks.KS_OPT_CLUSTER_SIZE, 8), (ks.KS_OPT_BLOCK_THREADS, 64)])):
        b, r = _gpu(ks, M, L, A, p, seed, S, **kw)
        assert_rows_equal(b, r, ids, eb, er, "packed4 %r" % (kw,))
    for init in (0, L - 1, 5):
        q = dict(p, init_price=init)
        eb, er = oracle_rows(oracle, q, L, 333, seed, ids, 40)
        b, r = _gpu(ks, M, L, 333, q, seed, 40)
        assert_rows_equal(b, r, ids, eb, er, "packed4 init_price=%d" % init)
    sim = ks.KsSim(2, L, 100, p, 0)
    with pytest.raises(ks.KsError):
        sim.ks_set_option(ks.KS_OPT_ATOMIC_MODE, 1)    # PACKED4 has plain atomics only
    sim.ks_destroy()


def test_packed4_full_size_c4_sampled_markets(ks, oracle):
    """C4 under PACKED4 at full size in the launch configuration bench.py --rng packed4 times;
    the oracle runs the 64 seeded sampled markets."""
    c = CONFIGS["C4"]
    p = packed4(c.params)
    b, r = _gpu(ks, c.M, c.L, c.A, p, c.seed, c.S)
    ids = sampled_markets(c.M, c.seed)
    eb, er = oracle_rows(oracle, p, c.L, c.A, c.seed, ids, c.S)
    assert_rows_equal(b, r, ids, eb, er, "C4 packed4")


# ------------------------------------------------------------------ per-step trace + SIV-J statistics
def _gpu_traced(ks, M, L, A, params, seed, runs, K, opts=()):
    import torch
    sim = ks.KsSim(M, L, A, params, seed)
    for o, v in opts:
        sim.ks_set_option(o, v)
    traces = []
    for S in runs:
        tr = torch.full((M, S, 2), -7, dtype=torch.int32, device="cuda")
        sim.ks_run_traced(S, tr)
        traces.append(tr)
    full = torch.cat(traces, dim=1).contiguous()
    st = ks.ks_trace_stats(full, M, full.shape[1], K)
    torch.cuda.synchronize()
    b, r = sim.books_to_host(), sim.stats_to_host()
    sim.ks_destroy()
    return b, r, full.cpu().numpy(), st.cpu().numpy()


def _assert_stats_close(got, exp, what, K):
    """The GPU forms every statistic as the quotient of two exact integers; the oracle evaluates
    the plain two-pass fp64 definitions.  Columns [0] volatility, [2] volume per step, [3] mean
    return: 1e-12 RELATIVE (north_star).  [1] excess kurtosis = m4/m2^2 - 3: 1e-12 relative to the
    kurtosis m4/m2^2 = exp + 3 >= 1, the quantity both sides compute before the constant is
    subtracted (a result near 0 carries the rounding of a number near 3).  The autocorrelations
    [4, 4+2K) are normalised to [-1, 1] and can be arbitrarily close to 0: 1e-12 ABSOLUTE
    (DESIGN.md 6.6)."""
    assert got.shape == exp.shape and got.shape[1] == 4 + 2 * K
    assert np.array_equal(np.isnan(got), np.isnan(exp)), what
    scale = np.abs(exp)
    scale[:, 1] = np.abs(exp[:, 1] + 3.0)
    scale[:, 4:] = 1.0
    m = ~np.isnan(exp)
    err = np.abs(got[m] - exp[m])
    assert np.all(err <= 1e-12 * scale[m]), "%s: worst err/tol %g" % (what, np.max(err / np.maximum(1e-12 * scale[m], 1e-300)))


@pytest.mark.parametrize("case", ["zi", "mix3", "packed4", "cluster", "long"])
def test_trace_and_return_statistics(ks, oracle, case):
    """the (price, Vmax) trace is bit-exact against the oracle's, tracing
    leaves the state bytes unchanged, traces of split runs concatenate, ragged step counts (not a
    multiple of the 32-entry staging buffer) flush completely, and the SIV-J statistics agree."""
    K = 20
    opts = ()
    if case == "zi":
        M, L, A, seed, p, runs = 37, 256, 700, 9, zi_params(16, 100), [45, 1, 32, 83]
    elif case == "mix3":
        M, L, A, seed, p, runs = 21, 1024, 900, 4, mix3_params(), [150]
    elif case == "packed4":
        M, L, A, seed, p, runs = 19, 512, 1001, 6, packed4(mix3_params()), [64, 37]
    elif case == "long":             # S = 10^5, the bound include/kineticsim.h states for ks_trace_stats (decoupled kernel)
        M, L, A, seed, p, runs = 3, 128, 64, 13, zi_params(8, 10), [100000]
    else:
        M, L, A, seed, p, runs = 9, 512, 600, 8, zi_params(32, 50), [70]
        opts = [(ks.KS_OPT_CLUSTER_SIZE, 4)]
    S = sum(runs)
    ids = np.arange(M)
    eb, er, et = oracle.run_markets_traced(p, L, A, seed, ids, S)
    b, r, tr, st = _gpu_traced(ks, M, L, A, p, seed, runs, K, opts)
    assert_rows_equal(b, r, ids, eb, er, "traced " + case)
    assert np.array_equal(tr, et), "trace differs from the oracle"
    exp = np.stack([oracle.trace_stats(et[i], K) for i in range(M)])
    _assert_stats_close(st, exp, "trace stats " + case, K)


def test_trace_stats_degenerate_series(ks, oracle):
    """Hand-made traces through ks_trace_stats alone: constant price (zero variance -> NaN),
    alternating +-1 returns (ACF (-1)^k (n-k)/n), one traced step (no returns), large moves near
    the int64 guard."""
    import torch
    K, S = 6, 101
    p = np.zeros((5, S, 2), dtype=np.int32)
    p[0, :, 0] = 77; p[0, :, 1] = 3
    p[1, :, 0] = 100 + (np.arange(S) % 2)
    p[2, :, 0] = np.arange(S) * 5
    p[3, :, 0] = np.where(np.arange(S) % 7 < 3, 32767, 0); p[3, :, 1] = 2 ** 31 - 1
    rng = np.random.default_rng(3)
    p[4, :, 0] = 500 + np.cumsum(rng.integers(-20, 21, size=S)); p[4, :, 1] = rng.integers(0, 1000, size=S)
    d = torch.from_numpy(p).cuda()
    got = ks.ks_trace_stats(d, 5, S, K).cpu().numpy()
    exp = np.stack([oracle.trace_stats(p[i], K) for i in range(5)])
    _assert_stats_close(got, exp, "degenerate", K)
    assert got[1, 0] == 1.0 and got[1, 1] == -2.0 and got[1, 4] == -(100 - 1) / 100
    one = ks.ks_trace_stats(d[:, :1, :].contiguous(), 5, 1, K).cpu().numpy()
    assert np.array_equal(one[:, 2], p[:, 0, 1].astype(np.float64)) and np.isnan(np.delete(one, 2, axis=1)).all()


# ------------------------------------------------------------------ the paper's own agent model
@pytest.mark.parametrize("alpha_mom", [0.0, 0.15, 0.7])
def test_paper_agent_model_matches_the_oracle(ks, oracle, alpha_mom):
    """SURVEY.md S8(f)-2 / DESIGN.md A24: mid-price reference (Eq.3) from the exact best quotes of
    the resting book, marketable orders at the grid boundary, parity makers, momentum on mid
    changes, classes by index ranges.  Several grid sizes (full-grid windows through
    clear_window<4>/<8> and the chunked scan), block sizes, split / launch-per-step runs, injected
    books whose best quotes lie far outside the active window, the trace."""
    import torch
    for (M, L, A, S, T, pm) in [(17, 128, 200, 120, 0, 0.05), (9, 256, 333, 60, 96, 0.2), (7, 2048, 500, 50, 0, 0.02),
                                (5, 64, 90, 80, 1024, 0.0), (6, 512, 64, 60, 32, 1.0)]:
        p = paper_params(A, alpha_mom, 0.15, delta=min(8, L // 8), p_mkt=pm)
        ids = np.arange(M)
        eb, er = oracle_rows(oracle, p, L, A, 5, ids, S)
        for kw in (dict(), dict(split=[1, S // 2, S - 1 - S // 2]), dict(stepwise=True), dict(opts=[(ks.KS_OPT_CLEAR_PATH, 1)])):
            opts = list(kw.pop("opts", [])) + [(ks.KS_OPT_BLOCK_THREADS, T)]
            b, r = _gpu(ks, M, L, A, p, 5, S, opts=opts, **kw)
            assert_rows_equal(b, r, ids, eb, er, "paper model L=%d alpha=%.2f %r" % (L, alpha_mom, kw))
    # injected books: crossed / one-sided / sparse far-away quotes
    M, L, A = 8, 1024, 150
    p = paper_params(A, alpha_mom, 0.15, delta=6, p_mkt=0.0)
    books = random_books(M, L, seed=3, max_qty=30, fill=0.01)
    books[0] = 0
    books[1, 1] = 0
    books[2] = 0; books[2, 0, 3] = 5; books[2, 1, 1000] = 5           # quotes far from the price
    books[3] = random_books(1, L, seed=9, fill=0.002, crossed=False)[0]
    eb0, er0 = oracle.init_state(M, L, -1, model=4)
    eb, er, et = oracle.run_markets_traced(p, L, A, 7, np.arange(M), 40, books, er0)
    sim = ks.KsSim(M, L, A, p, 7)
    sim.ks_write_books(torch.from_numpy(books).cuda())
    tr = torch.empty((M, 40, 2), dtype=torch.int32, device="cuda")
    sim.ks_run_traced(40, tr)
    b, r = sim.books_to_host(), sim.stats_to_host()
    assert_rows_equal(b, r, np.arange(M), eb, er, "paper model injected")
    assert np.array_equal(tr.cpu().numpy(), et)
    with pytest.raises(ks.KsError):
        sim.ks_set_option(ks.KS_OPT_CLUSTER_SIZE, 2)
    sim.ks_destroy()


def test_paper_agent_model_full_size_sampled_markets(ks, oracle):
    """Model 4 in the C4 shape (M = 65536 markets, L = 512, A = 4096; S = 200 so that the oracle,
    which scans the whole book for Eq.3 every step, stays in seconds) in the automatic launch plan:
    64 seeded sampled markets against the oracle, conservation on every market."""
    c = CONFIGS["C4"]
    S = 200
    p = paper_params(c.A, 0.15, 0.15, delta=32, qmax=100, half_spread=3, p_mkt=0.02)
    b, r = _gpu(ks, c.M, c.L, c.A, p, c.seed, S)
    ids = sampled_markets(c.M, c.seed, 64)
    eb, er = oracle_rows(oracle, p, c.L, c.A, c.seed, ids, S)
    assert_rows_equal(b, r, ids, eb, er, "model 4, C4 shape")
    r64 = r.astype(np.int64)
    tot = b.astype(np.int64).sum(axis=2)
    assert (b >= 0).all() and (r64[:, 0] == S).all()
    assert (r64[:, 10] == r64[:, 2] + tot[:, 0]).all() and (r64[:, 11] == r64[:, 2] + tot[:, 1]).all()


# ------------------------------------------------------------------ book injection / edge cases
def test_paper_worked_example_through_the_library(ks):
    """PAPER.md:315-354 (Eq.11-18) embedded at ticks 10..14 of an L=32 grid, A = 0: zero padding
    leaves p*, Vmax and the residual books unchanged."""
    ex = read_golden("paper_worked_example.txt")[0]
    books = np.zeros((3, 2, 32), dtype=np.int32)
    books[1, 0, 10:15] = ints(ex, "BUY"); books[1, 1, 10:15] = ints(ex, "SELL")
    b, r = _gpu(ks, 3, 32, 0, zi_params(1, 1), 0, 1, books=books)
    assert list(b[1, 0, 10:15]) == list(ints(ex, "new_bid")) and list(b[1, 1, 10:15]) == list(ints(ex, "new_ask"))
    assert b[1].sum() == ints(ex, "new_bid").sum() + ints(ex, "new_ask").sum()
    assert r[1, 12] == 10 + int(ex["pstar"][0]) and r[1, 2] == int(ex["vmax"][0]) and r[1, 1] == 1
    assert r[0, 1] == 0 and r[0, 12] == 16 and (b[0] == 0).all()          # empty market: no trade


@pytest.mark.parametrize("L,A,model", [(32, 0, "zi"), (64, 77, "zi"), (2048, 300, "mix3"), (4096, 0, "zi")])
def test_random_injected_books(ks, oracle, L, A, model):
    """Arbitrary (crossed, wide) resting books written with ks_write_books: the first step clears a
    window as wide as the grid (chunked general scan), later steps the narrow one."""
    M, S, seed = 9, 6, 12
    p = zi_params(min(8, L // 4), 10) if model == "zi" else mix3_params()
    books = random_books(M, L, seed=L + A, max_qty=40, fill=0.3)
    books[0] = 0                                   # empty market
    books[1, 1] = 0                                # one-sided market
    books[2] = random_books(1, L, seed=1, crossed=False)[0]
    eb0, er0 = oracle.init_state(M, L, -1)
    eb, er = oracle_rows(oracle, p, L, A, seed, np.arange(M), S, books=books, recs=er0)
    for clear in (0, 1):
        b, r = _gpu(ks, M, L, A, p, seed, S, books=books, opts=[(ks.KS_OPT_CLEAR_PATH, clear)])
        assert_rows_equal(b, r, np.arange(M), eb, er, "injected L=%d clear=%d" % (L, clear))


def test_price_pinned_to_grid_edge(ks, oracle):
    """init_price at the edges: clamped orders pile on ticks 0 / L-1 (A15) and the clamp path of
    the generator is exercised."""
    for init in (0, 63, 3):
        p = zi_params(8, 10, init_price=init)
        eb, er = oracle_rows(oracle, p, 64, 200, 5, np.arange(4), 50)
        b, r = _gpu(ks, 4, 64, 200, p, 5, 50)
        assert_rows_equal(b, r, np.arange(4), eb, er, "init_price=%d" % init)
    p = mix3_params(init_price=1)
    eb, er = oracle_rows(oracle, p, 128, 333, 6, np.arange(3), 40)
    b, r = _gpu(ks, 3, 128, 333, p, 6, 40)
    assert_rows_equal(b, r, np.arange(3), eb, er, "mix3 at the edge")


def test_max_grid_and_overflow_guards(ks, oracle):
    """L = 16384 (the single-CTA maximum); KS_ERR_OVERFLOW before a run that could pass 2^31."""
    p = zi_params(300, 7)
    eb, er = oracle_rows(oracle, p, 16384, 500, 3, np.arange(2), 12)
    b, r = _gpu(ks, 2, 16384, 500, p, 3, 12)
    assert_rows_equal(b, r, np.arange(2), eb, er, "L=16384")
    sim = ks.KsSim(1, 64, 4096, zi_params(8, 1 << 20), 0)
    with pytest.raises(ks.KsError) as e:
        sim.ks_run(1)
    assert e.value.status == ks.KS_ERR_OVERFLOW
    sim.ks_run(0)
    assert sim.stats_to_host()[0, 0] == 0
    sim.ks_destroy()


def test_run_to_run_determinism(ks):
    c = CONFIGS["C2"]
    a = _gpu(ks, 256, c.L, c.A, c.params, c.seed, 50)
    b = _gpu(ks, 256, c.L, c.A, c.params, c.seed, 50)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_debug_checks_build(ks):
    """compute-sanitizer is closed on this pool (profiles/r2_sanitizer.md); the library's own
    KS_DEBUG_CHECKS build stands in for it: every order address inside its target array, every
    clearing access inside the grid, no negative depth, and -- the phase structure of Alg.1
     -- exactly the step's orders in the book / histogram when the
    clearing warp starts.  All kernel families run under it (tests/sanitizer_cases.py, compared
    with the oracle); the negative control (barrier B1 dropped) must trap."""
    import os
    import subprocess
    import sys
    from paper_2606_21784_b200 import build
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for inject in (False, True):
        lib = build.DEBUG_INJECT_LIB if inject else build.DEBUG_LIB
        if build.debug_is_stale(lib):
            build.build_debug_checks(inject_race=inject)
    env = dict(os.environ, KINETICSIM_LIB=build.DEBUG_LIB)
    p = subprocess.run([sys.executable, os.path.join(root, "tests", "sanitizer_cases.py")], env=env, capture_output=True,
                       text=True, timeout=900)
    assert p.returncode == 0 and "all sanitizer cases ok" in p.stdout, p.stdout[-2000:] + p.stderr[-2000:]
    assert "KS_DEBUG_CHECKS failed" not in p.stdout + p.stderr
    env = dict(os.environ, KINETICSIM_LIB=build.DEBUG_INJECT_LIB)
    p = subprocess.run([sys.executable, os.path.join(root, "tests", "sanitizer_cases.py"), "c5"], env=env, capture_output=True,
                       text=True, timeout=900)
    assert p.returncode != 0 and "KS_DEBUG_CHECKS failed: orders in the book at B1" in p.stdout + p.stderr, \
        "the injected race was not caught: " + p.stdout[-1000:] + p.stderr[-1000:]


def test_random_shapes_in_the_automatic_plan(ks, oracle):
    """Seeded random shapes and parameters through WHATEVER plan the library picks (persistent, decoupled
    single-step, two steps per pass, the three-type decoupled path: `ks_plan_string` is recorded in
    the failure message), each also with the persistent kernel forced and with the decoupled kernel
    and two steps per pass forced: always the oracle's bytes.
    Shapes are drawn around the plan's thresholds (A = 128, 512, 1024, 1536; few or many markets; S
    odd, tiny, split)."""
    rng = np.random.default_rng(20261105)
    seen = set()
    for it in range(36):
        mix = it % 3 == 2
        L = int(rng.choice([64, 128, 256, 512, 1024]))
        A = int(rng.choice([0, 1, 31, 127, 128, 300, 511, 512, 700, 1023, 1024, 1535, 1536, 2000, 4100]))
        M = int(rng.choice([1, 2, 5, 37, 160, 700, 1300]))
        S = int(rng.choice([1, 2, 3, 5, 8, 17, 30]))
        if M * A * S > 6e6:
            M = max(1, int(6e6 // max(1, A * S)))
        if mix:
            p = dict(mix3_params(), noise_delta=int(rng.integers(0, min(64, L // 4))), noise_qmax=int(rng.integers(1, 60)),
                     maker_spread_max=int(rng.integers(1, 9)), maker_qty=int(rng.integers(1, 30)),
                     mom_delta=int(rng.integers(0, 12)), mom_qmax=int(rng.integers(1, 60)))
        else:
            p = zi_params(int(rng.integers(0, min(40, L // 4))), int(rng.integers(1, 120)))
        p["init_price"] = int(rng.choice([-1, 0, L - 1, L // 3]))
        seed = int(rng.integers(0, 2**40))
        ids = np.arange(M)
        eb, er = oracle_rows(oracle, p, L, A, seed, ids, S)
        split = None if S < 3 or it % 2 else [1, S - 2, 1]
        for forced in ((), ((ks.KS_OPT_PIPELINE, 1),), ((ks.KS_OPT_PIPELINE, 2), (ks.KS_OPT_STEP_PAIRS, 2))):
            sim = ks.KsSim(M, L, A, p, seed)
            for o, v in forced:
                sim.ks_set_option(o, v)
            plan = sim.ks_plan_string()
            seen.add(plan.split(" T=")[0] + (" pairs" if "steps_per_pass=2" in plan else "") + (" mix3" if "mix3" in plan else ""))
            for s_ in (split or [S]):
                sim.ks_run(s_)
            b, r = sim.books_to_host(), sim.stats_to_host()
            sim.ks_destroy()
            assert_rows_equal(b, r, ids, eb, er, "random shape %d: M=%d L=%d A=%d S=%d %s plan=%s" % (it, M, L, A, S, "mix3" if mix else "zi", plan))
    assert {"ks_decoupled_kernel", "ks_persistent_kernel", "ks_decoupled_kernel pairs", "ks_decoupled_kernel pairs mix3"} <= seen, seen
