"""Helpers for the tests: golden-file parser and two independent restatements of the clearing
definition (brute force over all ticks; greedy unit matching).  These live in the test tree, not
in oracle/: they are what the oracle is pinned AGAINST."""
import os

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLDEN = os.path.join(ROOT, "tests", "golden")


def read_golden(name):
    """Parse a tests/golden/*.txt fixture: '#' lines are comments (citations), blank lines
    separate records, 'key: v v v' lines are fields.  -> list of dict(key -> list of str)."""
    recs, cur = [], {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.rstrip("\n")
            if line.startswith("#"):
                continue
            if not line.strip():
                if cur:
                    recs.append(cur)
                    cur = {}
                continue
            k, v = line.split(":", 1)
            cur[k.strip()] = v.split()
    if cur:
        recs.append(cur)
    return recs




def ints(rec, key):
    return np.array([int(x) for x in rec[key]], dtype=np.int64)


def brute_force_price(bid, ask):
    """Eq.1-2 evaluated literally, O(L^2): for every p sum the bids at q >= p
    and the asks at q <= p; the price is the lowest p attaining the largest min(D, S).
    -> (pstar or -1, vmax, D, S)."""
    L = len(bid)
    D = [sum(int(bid[q]) for q in range(L) if q >= p) for p in range(L)]
    S = [sum(int(ask[q]) for q in range(L) if q <= p) for p in range(L)]
    V = [min(D[p], S[p]) for p in range(L)]
    vmax = max(V)
    pstar = V.index(vmax) if vmax > 0 else -1
    return pstar, vmax, D, S


def greedy_match(bid, ask):
    """Price-priority matching one lot at a time: repeatedly take the highest
    outstanding bid and the lowest outstanding ask; while bid tick >= ask tick, trade
    min(remaining) lots.  Stops when the book is uncrossed.  -> (volume, new_bid, new_ask).
    Knows nothing of cumulative profiles or of p*."""
    b = [int(x) for x in bid]
    a = [int(x) for x in ask]
    L = len(b)
    vol = 0
    hi, lo = L - 1, 0
    while True:
        while hi >= 0 and b[hi] == 0:
            hi -= 1
        while lo < L and a[lo] == 0:
            lo += 1
        if hi < 0 or lo >= L or hi < lo:
            break
        x = min(b[hi], a[lo])
        b[hi] -= x
        a[lo] -= x
        vol += x
    return vol, np.array(b, dtype=np.int64), np.array(a, dtype=np.int64)


def oracle_rows(oracle, params, L, A, seed, ids, S, books=None, recs=None, threads=None):
    """Run the (single-threaded) oracle on the markets `ids`, one independent oracle call per
    host thread over disjoint id ranges (markets are independent; ctypes releases the GIL)."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    ids = np.asarray(ids, dtype=np.uint32)
    n = len(ids)
    threads = max(1, min(threads or (os.cpu_count() or 1), n))
    cuts = np.linspace(0, n, threads + 1).astype(int)

    def job(k):
        lo, hi = cuts[k], cuts[k + 1]
        if lo == hi:
            return None
        b = None if books is None else books[lo:hi]
        r = None if recs is None else recs[lo:hi]
        return oracle.run_markets(params, L, A, seed, ids[lo:hi], S, b, r)

    with ThreadPoolExecutor(threads) as ex:
        parts = [p for p in ex.map(job, range(threads)) if p is not None]
    return np.concatenate([p[0] for p in parts]), np.concatenate([p[1] for p in parts])


def assert_rows_equal(gpu_books, gpu_recs, ids, exp_books, exp_recs, what=""):
    """Bit-exact comparison of the sampled rows: books, prices, every integer sum and the hash."""
    ids = np.asarray(ids, dtype=np.int64)
    gb, gr = gpu_books[ids], gpu_recs[ids]
    if not np.array_equal(gr, exp_recs):
        bad = np.argwhere(gr != exp_recs)
        i, f = bad[0]
        raise AssertionError("%s: record mismatch at market %d field %d: gpu %d oracle %d (%d mismatches)"
                             % (what, ids[i], f, gr[i, f], exp_recs[i, f], len(bad)))
    if not np.array_equal(gb, exp_books):
        bad = np.argwhere(gb != exp_books)
        i, s, p = bad[0]
        raise AssertionError("%s: book mismatch at market %d side %d tick %d: gpu %d oracle %d (%d mismatches)"
                             % (what, ids[i], s, p, gb[i, s, p], exp_books[i, s, p], len(bad)))


def sass_innermost_loops(sass_text, function_substring):
    """Innermost loops of one kernel in `cuobjdump -sass` output: a loop is the address range of a
    backward branch; -> list of dict(n=instructions, atoms=ATOMS count, mults=IMAD.WIDE.U32 +
    IMAD.HI.U32 count, lop3=...) for the loops that contain no other loop."""
    import re
    bodies = [p for p in sass_text.split("Function : ") if function_substring in p.split("\n", 1)[0]]
    assert len(bodies) == 1, "%d kernels match %r" % (len(bodies), function_substring)
    ins = []
    for line in bodies[0].splitlines():
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", line)
        if m:
            ins.append((int(m.group(1), 16), m.group(2)))
    loops = []
    for addr, text in ins:
        m = re.search(r"\bBRA\b.*?0x([0-9a-f]+)", text)
        if m and int(m.group(1), 16) <= addr:
            loops.append((int(m.group(1), 16), addr))
    inner = [(lo, hi) for lo, hi in loops if not any((l2, h2) != (lo, hi) and lo <= l2 and h2 <= hi for l2, h2 in loops)]
    out = []
    for lo, hi in inner:
        body = [t for a, t in ins if lo <= a <= hi]
        out.append(dict(n=len(body), atoms=sum("ATOMS" in t for t in body),
                        mults=sum("IMAD.WIDE.U32" in t or "IMAD.HI.U32" in t for t in body),
                        lop3=sum("LOP3" in t for t in body)))
    return out
