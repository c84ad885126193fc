"""ctypes wrapper around oracle/ks_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It holds no arithmetic of the method: it builds the C file with gcc,
marshals numpy arrays in and out, and nothing else.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ks_oracle.c")
_LIB = os.path.join(_HERE, "libks_oracle.so")
_lock = threading.Lock()
_lib = None

PARAM_FIELDS = ("model", "noise_delta", "noise_qmax", "maker_spread_max", "maker_qty",
                "mom_delta", "mom_qmax", "init_price", "paper_n_mom", "paper_n_maker", "paper_pmkt_q16")

# record field names, in order
REC_FIELDS = ("steps", "n_trades", "sum_vol", "sum_px", "sum_px2", "sum_pxvol", "sum_ret",
              "sum_ret2", "sum_ret3", "sum_ret4", "sub_buy", "sub_sell", "last", "prev",
              "traj_hash", "n_orders")
DERIVED_FIELDS = ("mean_px", "vwap", "vol_per_step", "ret_mean", "ret_var", "excess_kurtosis")


class KoParams(C.Structure):
    _fields_ = [(n, C.c_int32) for n in PARAM_FIELDS]


def build(force: bool = False) -> str:
    """Compile ks_oracle.c into libks_oracle.so with gcc (-O2, no fast-math)."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + ".tmp.%d" % os.getpid()
            subprocess.check_call(["gcc", "-O2", "-std=c99", "-Wall", "-Wextra", "-shared", "-fPIC",
                                   "-fvisibility=hidden", "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u32p, i32p, i64p = C.POINTER(C.c_uint32), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
        L.ko_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.ko_philox4x32_10.restype = None
        L.ko_gen_orders.argtypes = [C.POINTER(KoParams), C.c_int32, C.c_int32, C.c_int32, C.c_uint64,
                                    C.c_uint32, C.c_uint32, C.c_uint32, i32p, i32p, i32p]
        L.ko_gen_orders.restype = C.c_int32
        L.ko_clear_step.argtypes = [i64p, i64p, C.c_int32, i64p, i64p, i64p, i32p, i64p]
        L.ko_clear_step.restype = None
        L.ko_init_record.argtypes = [i64p, C.c_int32, C.c_int32]
        L.ko_init_record.restype = None
        L.ko_init_record_paper.argtypes = [i64p, C.c_int32, C.c_int32]
        L.ko_init_record_paper.restype = None
        L.ko_gen_orders_paper.argtypes = [C.POINTER(KoParams), C.c_int32, C.c_int32, C.c_int32, C.c_uint64,
                                          C.c_uint32, C.c_uint32, C.c_uint32, C.c_int32, i32p, i32p, i32p]
        L.ko_gen_orders_paper.restype = C.c_int32
        L.ko_run_markets.argtypes = [C.POINTER(KoParams), C.c_int32, C.c_int32, C.c_uint64, u32p,
                                     C.c_int32, C.c_int64, i32p, i64p]
        L.ko_run_markets.restype = C.c_int32
        L.ko_run_markets_traced.argtypes = [C.POINTER(KoParams), C.c_int32, C.c_int32, C.c_uint64, u32p,
                                            C.c_int32, C.c_int64, i32p, i64p, i32p]
        L.ko_run_markets_traced.restype = C.c_int32
        L.ko_trace_stats.argtypes = [i32p, C.c_int64, C.c_int32, C.POINTER(C.c_double)]
        L.ko_trace_stats.restype = None
        L.ko_derived.argtypes = [i64p, C.POINTER(C.c_double)]
        L.ko_derived.restype = None
        _lib = L
    return _lib


def _params(p: dict) -> KoParams:
    return KoParams(*[int(p.get(n, 0)) for n in PARAM_FIELDS])


def _ptr(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().ko_philox4x32_10(_ptr(c, C.c_uint32), _ptr(k, C.c_uint32), _ptr(out, C.c_uint32))
    return out


def gen_orders(params: dict, L: int, last: int, prev: int, seed: int, m: int, t: int, a: int):
    """-> list of (side, tick, qty); side 0 = bid (buy), 1 = ask (sell)."""
    side = np.zeros(2, np.int32); tick = np.zeros(2, np.int32); qty = np.zeros(2, np.int32)
    P = _params(params)
    n = lib().ko_gen_orders(C.byref(P), L, last, prev, seed, m, t, a,
                            _ptr(side, C.c_int32), _ptr(tick, C.c_int32), _ptr(qty, C.c_int32))
    return [(int(side[i]), int(tick[i]), int(qty[i])) for i in range(n)]


def clear_step(bid, ask):
    """Clear one combined book.  -> dict(D, S, V, pstar, vmax, new_bid, new_ask); pstar = -1 if no trade."""
    b = np.asarray(bid, dtype=np.int64).copy()
    a = np.asarray(ask, dtype=np.int64).copy()
    L = b.shape[0]
    assert a.shape == (L,) and L >= 1
    D = np.zeros(L, np.int64); S = np.zeros(L, np.int64); V = np.zeros(L, np.int64)
    ps = C.c_int32(0); vm = C.c_int64(0)
    lib().ko_clear_step(_ptr(b, C.c_int64), _ptr(a, C.c_int64), L, _ptr(D, C.c_int64),
                        _ptr(S, C.c_int64), _ptr(V, C.c_int64), C.byref(ps), C.byref(vm))
    return dict(D=D, S=S, V=V, pstar=int(ps.value), vmax=int(vm.value), new_bid=b, new_ask=a)


def init_state(n: int, L: int, init_price: int = -1, model: int = 0):
    """Fresh state for n markets: (books int32 [n][2][L] = 0, recs int64 [n][16]).  Model 4 keeps
    the doubled previous mid in f[13]."""
    books = np.zeros((n, 2, L), dtype=np.int32)
    recs = np.zeros((n, 16), dtype=np.int64)
    for i in range(n):
        (lib().ko_init_record_paper if model == 4 else lib().ko_init_record)(_ptr(recs[i], C.c_int64), L, init_price)
    return books, recs


def gen_orders_paper(params: dict, L: int, mid2: int, mid2_prev: int, seed: int, m: int, t: int, a: int, A: int):
    """Model 4 -> (side, tick, qty)."""
    side = C.c_int32(0); tick = C.c_int32(0); qty = C.c_int32(0)
    P = _params(params)
    lib().ko_gen_orders_paper(C.byref(P), L, mid2, mid2_prev, seed, m, t, a, A,
                              C.byref(side), C.byref(tick), C.byref(qty))
    return int(side.value), int(tick.value), int(qty.value)


def run_markets(params: dict, L: int, A: int, seed: int, ids, S: int, books=None, recs=None):
    """Run S steps of the markets with global ids `ids`, continuing from (books, recs) (fresh if None).

    Returns (books, recs) -- new arrays; inputs are not modified.  Raises on an internal
    consistency failure of the oracle (negative depth, buy/sell volume mismatch, 2^31 overflow).
    """
    ids = np.ascontiguousarray(np.asarray(ids, dtype=np.uint32))
    n = ids.shape[0]
    if books is None:
        books, recs = init_state(n, L, int(params["init_price"]), int(params["model"]))
    else:
        books = np.ascontiguousarray(books, dtype=np.int32).copy()
        recs = np.ascontiguousarray(recs, dtype=np.int64).copy()
    assert books.shape == (n, 2, L) and recs.shape == (n, 16)
    P = _params(params)
    rc = lib().ko_run_markets(C.byref(P), L, A, seed, _ptr(ids, C.c_uint32), n, S,
                              _ptr(books, C.c_int32), _ptr(recs, C.c_int64))
    if rc != 0:
        raise RuntimeError("oracle consistency assertion failed, code %d" % rc)
    return books, recs


def run_markets_traced(params: dict, L: int, A: int, seed: int, ids, S: int, books=None, recs=None):
    """run_markets that also returns trace int32 [n][S][2] = (price after the step, Vmax)."""
    ids = np.ascontiguousarray(np.asarray(ids, dtype=np.uint32))
    n = ids.shape[0]
    if books is None:
        books, recs = init_state(n, L, int(params["init_price"]), int(params["model"]))
    else:
        books = np.ascontiguousarray(books, dtype=np.int32).copy()
        recs = np.ascontiguousarray(recs, dtype=np.int64).copy()
    trace = np.zeros((n, S, 2), dtype=np.int32)
    P = _params(params)
    rc = lib().ko_run_markets_traced(C.byref(P), L, A, seed, _ptr(ids, C.c_uint32), n, S,
                                     _ptr(books, C.c_int32), _ptr(recs, C.c_int64), _ptr(trace, C.c_int32))
    if rc != 0:
        raise RuntimeError("oracle consistency assertion failed, code %d" % rc)
    return books, recs, trace


def trace_stats(trace, K: int):
    """trace int32 [S][2] of one market -> float64 [4 + 2K] (see ko_trace_stats)."""
    t = np.ascontiguousarray(trace, dtype=np.int32)
    out = np.zeros(4 + 2 * K, dtype=np.float64)
    lib().ko_trace_stats(_ptr(t, C.c_int32), t.shape[0], K, _ptr(out, C.c_double))
    return out


def derived(rec):
    r = np.ascontiguousarray(rec, dtype=np.int64)
    out = np.zeros(6, dtype=np.float64)
    lib().ko_derived(_ptr(r, C.c_int64), _ptr(out, C.c_double))
    return out
