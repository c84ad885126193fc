"""The two exactness arguments the CUDA clearing rests on, checked by brute
force in numpy against the plain full-grid definition (Eq.1-2, lowest-tick
tie-break, strict price priority) on random small books -- no GPU, no oracle code:
  1. scanning any window [lo, hi] that contains every ask's lowest tick and every bid's highest
     tick gives the full-grid price, volume and residual book;
  2. ExtDepth: depth at the edge ticks (marketable buys at L-1, sells at 0) may be folded into the
     window's profiles as two constants iff  ext_b <= S[top]  and  (ext_a == 0 or (ext_a <= D[base]
     and Vmax > ext_a)); then the edge ticks end empty."""
import numpy as np


def full_grid(bid, ask):
    D = np.cumsum(bid[::-1])[::-1]
    S = np.cumsum(ask)
    V = np.minimum(D, S)
    vm = int(V.max())
    if vm == 0:
        return 0, -1, bid.copy(), ask.copy()
    p = int(np.argmax(V))                                   # first maximum = lowest tick
    return vm, p, np.minimum(bid, np.maximum(0, D - vm)), np.minimum(ask, np.maximum(0, S - vm))


def window(bid, ask, lo, hi, eb=0, ea=0):
    wb, wa = bid[lo:hi + 1], ask[lo:hi + 1]
    D = np.cumsum(wb[::-1])[::-1] + eb
    S = np.cumsum(wa) + ea
    V = np.minimum(D, S)
    v = int(V.max())
    ok = eb <= S[-1] and (ea == 0 or (ea <= D[0] and v > ea))
    nb, na = bid.copy(), ask.copy()
    if v > 0:
        nb[lo:hi + 1] = np.minimum(wb, np.maximum(0, D - v))
        na[lo:hi + 1] = np.minimum(wa, np.maximum(0, S - v))
    return ok, v, (lo + int(np.argmax(V)) if v > 0 else -1), nb, na


def _random_book(rng, L, lo, hi):
    """bids anywhere at ticks <= hi, asks anywhere at ticks >= lo: [lo, hi] contains amin and bmax."""
    bid, ask = np.zeros(L, dtype=np.int64), np.zeros(L, dtype=np.int64)
    m = rng.random(L) < 0.3
    bid[:hi + 1] = (rng.integers(1, 6, L) * m)[:hi + 1]
    m = rng.random(L) < 0.3
    ask[lo:] = (rng.integers(1, 6, L) * m)[lo:]
    return bid, ask


def test_any_window_containing_amin_and_bmax_is_exact():
    rng = np.random.default_rng(7)
    for _ in range(20000):
        L = 24
        lo = int(rng.integers(0, 10)); hi = int(rng.integers(lo + 1, L))
        bid, ask = _random_book(rng, L, lo, hi)
        vm, p, nb, na = full_grid(bid, ask)
        _, v, pw, wb, wa = window(bid, ask, lo, hi)
        assert (v, pw) == (vm, p) and (wb == nb).all() and (wa == na).all()


def test_ext_depth_condition_is_exact_and_not_vacuous():
    rng = np.random.default_rng(1)
    taken = refused = 0
    for _ in range(40000):
        L = 32
        lo = int(rng.integers(3, 12)); hi = int(rng.integers(lo + 3, 28))
        bid, ask = _random_book(rng, L, lo, hi)
        bid[L - 1] = 0; ask[0] = 0
        eb = int(rng.integers(1, 12)) if rng.random() < 0.7 else 0
        ea = int(rng.integers(1, 12)) if rng.random() < 0.7 else 0
        if eb == 0 and ea == 0:
            continue
        fb, fa = bid.copy(), ask.copy()
        fb[L - 1] += eb; fa[0] += ea
        vm, p, nb, na = full_grid(fb, fa)
        ok, v, pw, wb, wa = window(bid, ask, lo, hi, eb, ea)
        if not ok:
            refused += 1
            continue
        taken += 1
        assert (v, pw) == (vm, p)
        assert (wb == nb).all() and (wa == na).all()        # in particular nb[L-1] == 0 and na[0] == 0
    assert taken > 10000 and refused > 1000
    # the tie case that forces the strict Vmax > ext_a: only the marketable sells cross
    bid = np.zeros(16, dtype=np.int64); ask = np.zeros(16, dtype=np.int64)
    bid[8] = 5; ask[10] = 4; ask[0] = 3
    vm, p, _, _ = full_grid(bid, ask)
    assert (vm, p) == (3, 0)                                # the lowest tick attaining Vmax is tick 0 itself
    ask0 = ask.copy(); ask0[0] = 0
    assert window(bid, ask0, 6, 12, 0, 3)[0] is False
