"""Small runs of every kernel family for compute-sanitizer (racecheck / synccheck / memcheck):

    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py [case ...]

Each case goes through the C ABI and is compared with the oracle, so a hazard that changes a byte
fails here too.  Sizes are tiny because the sanitizer serialises the GPU.  Cases (SURVEY.md S4(4),
Alg.1's phase structure PAPER.md:143-176, 200-212):
  c1          C1 in the automatic plan (ks_decoupled_kernel: named barriers, two-step look-ahead)
  pairs       the two-steps-per-pass decoupled kernel (groups of ring slots handed over together), odd and split S
  mix3pairs   the three-type population under the decoupled kernel (relative maker / momentum bins)
  c5          a shrunk C5 (M=4, L=4096, A=1500, S=20, MIX3): ks_persistent_kernel, several warps, two barriers
  t32         one warp per market (T = 32): the barrier-light path C4 runs
  cluster     C = 4 CTAs per market, L = 1024: DSMEM reductions, barrier.cluster
  paper       model 4 with P_mkt > 0: the same-value flag writes s_mkt
  traced      ks_run_traced + ks_trace_stats
  packed      PACKED4 draws, ragged A
  generic     forced chunked scan + injected crossed books
  attach      checkpoint: run, attach a new handle, run
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import torch  # noqa: E402

from oracle import ks_oracle  # noqa: E402
from paper_2606_21784_b200 import binding as ks  # noqa: E402
from paper_2606_21784_b200.workloads import CONFIGS, mix3_params, packed4, paper_params, random_books, zi_params  # noqa: E402


def check(name, M, L, A, p, seed, S, opts=(), books=None, split=None):
    sim = ks.KsSim(M, L, A, p, seed)
    for o, v in opts:
        sim.ks_set_option(o, v)
    if books is not None:
        sim.ks_write_books(torch.from_numpy(np.ascontiguousarray(books)).cuda())
    for s in (split or [S]):
        sim.ks_run(s)
    b, r = sim.books_to_host(), sim.stats_to_host()
    sim.ks_destroy()
    recs0 = None if books is None else ks_oracle.init_state(M, L, int(p["init_price"]), int(p["model"]))[1]
    eb, er = ks_oracle.run_markets(p, L, A, seed, np.arange(M), S, books, recs0)
    assert np.array_equal(b, eb) and np.array_equal(r, er), name
    print("%s ok" % name, flush=True)


def c1():
    c = CONFIGS["C1"]
    check("c1", c.M, c.L, c.A, c.params, c.seed, c.S)
    check("c1 decoupled 3 markets", 3, 128, 512, zi_params(8, 10), 2, 40, opts=[(ks.KS_OPT_PIPELINE, 2)])


def pairs():
    opts = [(ks.KS_OPT_PIPELINE, 2), (ks.KS_OPT_STEP_PAIRS, 2)]
    check("pairs C2 shape, odd S", 9, 256, 1024, zi_params(16, 100), 1, 41, opts=opts)
    check("pairs T=96 split", 5, 512, 1500, zi_params(32, 100), 3, 30, opts=opts + [(ks.KS_OPT_BLOCK_THREADS, 96)], split=[1, 4, 25])


def mix3pairs():
    opts = [(ks.KS_OPT_PIPELINE, 2), (ks.KS_OPT_BLOCK_THREADS, 160)]
    check("mix3 decoupled, odd S", 5, 1024, 1541, mix3_params(), 4, 23, opts=opts)
    check("mix3 decoupled at the grid edge", 3, 256, 700, dict(mix3_params(), init_price=2), 4, 20, opts=opts, split=[3, 17])


def c5():
    check("c5 shrunk", 4, 4096, 1500, mix3_params(), 4, 20)
    check("c5 shrunk T=128", 4, 4096, 1500, mix3_params(), 4, 20, opts=[(ks.KS_OPT_BLOCK_THREADS, 128)])


def t32():
    check("t32", 6, 512, 700, zi_params(32, 100), 3, 30, opts=[(ks.KS_OPT_BLOCK_THREADS, 32), (ks.KS_OPT_PIPELINE, 1)])


def cluster():
    check("cluster C=4", 3, 1024, 900, mix3_params(), 7, 20, opts=[(ks.KS_OPT_CLUSTER_SIZE, 4)])
    check("cluster C=2 zi", 2, 1024, 400, zi_params(16, 100), 7, 20, opts=[(ks.KS_OPT_CLUSTER_SIZE, 2)])


def paper():
    check("paper", 4, 256, 600, paper_params(600, 0.15, 0.15, p_mkt=0.05), 5, 30)
    check("paper T=64", 4, 128, 200, paper_params(200, 0.3, 0.15, p_mkt=0.2), 5, 30, opts=[(ks.KS_OPT_BLOCK_THREADS, 64)])


def traced():
    M, L, A, S, K = 3, 128, 300, 70, 5
    p = zi_params(8, 10)
    sim = ks.KsSim(M, L, A, p, 9)
    tr = torch.zeros((M, S, 2), dtype=torch.int32, device="cuda")
    sim.ks_run_traced(S, tr)
    out = ks.ks_trace_stats(tr, M, S, K)
    torch.cuda.synchronize()
    r = sim.stats_to_host()
    sim.ks_destroy()
    _, er, etr = ks_oracle.run_markets_traced(p, L, A, 9, np.arange(M), S)
    assert np.array_equal(r, er) and np.array_equal(tr.cpu().numpy(), etr), "traced"
    assert np.isfinite(out.cpu().numpy()[:, 2]).all()
    print("traced ok", flush=True)


def packed():
    check("packed", 5, 256, 1001, packed4(zi_params(16, 100)), 9, 30)
    check("packed mix3", 3, 512, 1003, packed4(mix3_params()), 9, 20)


def generic():
    books = random_books(3, 256, 11, crossed=True)
    check("generic", 3, 256, 300, zi_params(16, 100), 9, 20, opts=[(ks.KS_OPT_CLEAR_PATH, 1)], books=books)


def attach():
    M, L, A, p, seed = 3, 128, 300, zi_params(8, 10), 12
    sim = ks.KsSim(M, L, A, p, seed)
    sim.ks_run(15)
    torch.cuda.synchronize()
    sim2 = ks.KsSim(M, L, A, p, seed, state=sim.state, attach=True)
    sim2.ks_run(10)
    b, r = sim2.books_to_host(), sim2.stats_to_host()
    sim2.ks_destroy(); sim.ks_destroy()
    eb, er = ks_oracle.run_markets(p, L, A, seed, np.arange(M), 25)
    assert np.array_equal(b, eb) and np.array_equal(r, er), "attach"
    print("attach ok", flush=True)


CASES = dict(c1=c1, pairs=pairs, mix3pairs=mix3pairs, c5=c5, t32=t32, cluster=cluster, paper=paper, traced=traced, packed=packed, generic=generic, attach=attach)

if __name__ == "__main__":
    ks.load()
    for n in (sys.argv[1:] or list(CASES)):
        CASES[n]()
    print("all sanitizer cases ok")
