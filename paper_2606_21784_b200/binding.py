"""Thin Python binding over the C ABI of libkineticsim.so (include/kineticsim.h) and of
libkineticsim_bench.so (include/kineticsim_bench.h: the launch-per-step ablation and the roofline
microbenchmarks): same names, argument marshalling only.  Every step of the hot path
runs in the CUDA kernels behind these calls; torch is used for device memory and streams only.

There is NO fallback: if the library is missing or was not built, `load()` raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkineticsim.so")
BENCH_LIB_PATH = os.path.join(_HERE, "libkineticsim_bench.so")

KS_OK, KS_ERR_INVALID_ARG, KS_ERR_UNSUPPORTED, KS_ERR_OVERFLOW, KS_ERR_CUDA, KS_ERR_NOMEM = 0, -1, -2, -3, -4, -5
KS_OPT_BLOCK_THREADS, KS_OPT_ATOMIC_MODE, KS_OPT_CLEAR_PATH, KS_OPT_CLUSTER_SIZE, KS_OPT_PIPELINE, KS_OPT_REL_COLUMNS, KS_OPT_RING_DEPTH, KS_OPT_STEP_PAIRS = 0, 1, 2, 3, 4, 5, 6, 7

PARAM_FIELDS = ("model", "noise_delta", "noise_qmax", "maker_spread_max", "maker_qty", "mom_delta",
                "mom_qmax", "init_price", "paper_n_mom", "paper_n_maker", "paper_pmkt_q16")
REC_FIELDS = ("steps", "n_trades", "sum_vol", "sum_px", "sum_px2", "sum_pxvol", "sum_ret", "sum_ret2",
              "sum_ret3", "sum_ret4", "sub_buy", "sub_sell", "last", "prev", "traj_hash", "n_orders")
DERIVED_FIELDS = ("mean_px", "vwap", "vol_per_step", "ret_mean", "ret_var", "excess_kurtosis")

# every symbol the two headers declare (tests check that each library exports exactly these)
EXPORTS = ("ks_state_bytes", "ks_create", "ks_create_ex", "ks_attach", "ks_run", "ks_read_books", "ks_read_stats",
           "ks_write_books", "ks_run_traced", "ks_trace_stats", "ks_set_option", "ks_derive_stats", "ks_destroy", "ks_last_error",
           "ks_launch_count", "ks_error_state", "ks_plan_string", "ks_depth_bound_static")
KS_DEPTH_BOUND_STATIC_MAX_M = 65536
BENCH_EXPORTS = ("ks_run_stepwise", "ks_bench_smem_atomic", "ks_bench_generate_only", "ks_bench_int_pipe")


class KsAgentParams(C.Structure):
    _fields_ = [(n, C.c_int32) for n in PARAM_FIELDS]


class KsError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__("kineticsim status %d: %s" % (status, text))
        self.status = status


_lib = None
_bench = None


def load_bench():
    """dlopen libkineticsim_bench.so (after the product library it is linked against)."""
    global _bench
    if _bench is not None:
        return _bench
    load()
    if not os.path.exists(BENCH_LIB_PATH):
        raise RuntimeError("libkineticsim_bench.so is not built (%s); run `python -m paper_2606_21784_b200.build`"
                           % BENCH_LIB_PATH)
    B = C.CDLL(BENCH_LIB_PATH)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    pp, pd = C.POINTER(KsAgentParams), C.POINTER(dbl)
    B.ks_run_stepwise.argtypes = [vp, i64, vp]; B.ks_run_stepwise.restype = i32
    B.ks_bench_smem_atomic.argtypes = [i32, i32, i32, i32, i32, i32, i32, i32, vp, pd, pd]
    B.ks_bench_smem_atomic.restype = i32
    B.ks_bench_generate_only.argtypes = [pp, i32, i32, i32, i64, i32, i32, i32, vp, pd, pd]
    B.ks_bench_generate_only.restype = i32
    B.ks_bench_int_pipe.argtypes = [i32, i32, i32, i32, i32, i32, vp, pd, pd]
    B.ks_bench_int_pipe.restype = i32
    _bench = B
    return B


def load():
    """dlopen libkineticsim.so and declare the prototypes.  Raises if the library is absent."""
    global _lib
    if _lib is not None:
        return _lib
    # KINETICSIM_LIB selects another build of the SAME CUDA library (the KS_DEBUG_CHECKS build); it is
    # not a fallback: the path must exist
    path = os.environ.get("KINETICSIM_LIB") or LIB_PATH
    if not os.path.exists(path):
        raise RuntimeError("libkineticsim.so is not built (%s); run `python -m paper_2606_21784_b200.build` "
                           "or __graft_entry__.build() -- there is no CPU fallback" % path)
    L = C.CDLL(path, mode=C.RTLD_GLOBAL)
    vp, i32, i64, u64, u32, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_uint32, C.c_double
    pp = C.POINTER(KsAgentParams)
    L.ks_state_bytes.argtypes = [i32, i32]; L.ks_state_bytes.restype = C.c_size_t
    L.ks_create.argtypes = [C.POINTER(vp), i32, i32, i32, pp, u64, vp, vp]; L.ks_create.restype = i32
    L.ks_create_ex.argtypes = [C.POINTER(vp), i32, i32, i32, pp, u64, u32, vp, vp]; L.ks_create_ex.restype = i32
    L.ks_run.argtypes = [vp, i64, vp]; L.ks_run.restype = i32
    L.ks_attach.argtypes = [C.POINTER(vp), i32, i32, i32, pp, u64, u32, vp, vp]; L.ks_attach.restype = i32
    L.ks_run_traced.argtypes = [vp, i64, vp, vp]; L.ks_run_traced.restype = i32
    L.ks_trace_stats.argtypes = [vp, i32, i64, i32, vp, vp]; L.ks_trace_stats.restype = i32
    L.ks_read_books.argtypes = [vp, vp, vp]; L.ks_read_books.restype = i32
    L.ks_read_stats.argtypes = [vp, vp, vp]; L.ks_read_stats.restype = i32
    L.ks_write_books.argtypes = [vp, vp, vp]; L.ks_write_books.restype = i32
    L.ks_set_option.argtypes = [vp, i32, i32]; L.ks_set_option.restype = i32
    L.ks_derive_stats.argtypes = [vp, vp, i64]; L.ks_derive_stats.restype = None
    L.ks_error_state.argtypes = [vp]; L.ks_error_state.restype = i32
    L.ks_plan_string.argtypes = [vp, C.c_char_p, C.c_size_t]; L.ks_plan_string.restype = i32
    L.ks_destroy.argtypes = [vp]; L.ks_destroy.restype = None
    L.ks_last_error.argtypes = []; L.ks_last_error.restype = C.c_char_p
    L.ks_launch_count.argtypes = []; L.ks_launch_count.restype = i64
    L.ks_depth_bound_static.argtypes = [vp, i32, i32, vp, vp]; L.ks_depth_bound_static.restype = i32
    _lib = L
    return L


def _check(status: int):
    if status != KS_OK:
        raise KsError(status, (load().ks_last_error() or b"").decode())


def _params(p: dict) -> KsAgentParams:
    return KsAgentParams(*[int(p.get(n, 0)) for n in PARAM_FIELDS])


def _stream_ptr(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _ptr_of(x) -> int:
    """Raw pointer of a torch tensor (device or pinned host) or a numpy array."""
    if isinstance(x, np.ndarray):
        assert x.flags["C_CONTIGUOUS"]
        return x.ctypes.data
    assert x.is_contiguous()
    return x.data_ptr()


def ks_state_bytes(M: int, L: int) -> int:
    return int(load().ks_state_bytes(M, L))


def ks_last_error() -> str:
    return (load().ks_last_error() or b"").decode()


def ks_launch_count() -> int:
    return int(load().ks_launch_count())


def ks_derive_stats(recs: np.ndarray) -> np.ndarray:
    """recs int64 [n][16] (host) -> float64 [n][6] (DERIVED_FIELDS)."""
    recs = np.ascontiguousarray(recs, dtype=np.int64).reshape(-1, 16)
    out = np.zeros((recs.shape[0], 6), dtype=np.float64)
    load().ks_derive_stats(recs.ctypes.data, out.ctypes.data, recs.shape[0])
    return out


class KsSim:
    """Owns the ks_sim handle and (unless one is passed in) the torch uint8 state tensor."""

    def __init__(self, M: int, L: int, A: int, params: dict, seed: int, market_base: int = 0,
                 state=None, stream=None, device="cuda:0", attach: bool = False):
        """attach=False: ks_create_ex (enqueues the initialisation of `state`).  attach=True:
        ks_attach -- adopt the checkpoint already in `state` (books, prices, step counter, sums)."""
        import torch
        lib = load()
        self.M, self.L, self.A = M, L, A
        nbytes = ks_state_bytes(M, L)
        if nbytes == 0:
            raise KsError(KS_ERR_INVALID_ARG, "ks_state_bytes rejected M=%d L=%d" % (M, L))
        assert state is not None or not attach, "ks_attach needs the state buffer that holds the checkpoint"
        if state is None:
            state = torch.empty(nbytes, dtype=torch.uint8, device=device)
        assert state.is_cuda and state.numel() >= nbytes
        self.state = state
        self._h = C.c_void_p(None)
        P = _params(params)
        with torch.cuda.device(state.device):      # the library records the current device in the handle
            _check((lib.ks_attach if attach else lib.ks_create_ex)(C.byref(self._h), M, L, A, C.byref(P), seed, market_base,
                                                                  state.data_ptr(), _stream_ptr(stream)))

    # -- the C ABI, same names -------------------------------------------------------------
    def ks_run(self, S: int, stream=None):
        _check(load().ks_run(self._h, S, _stream_ptr(stream)))

    def ks_run_stepwise(self, S: int, stream=None):
        load()
        _check(load_bench().ks_run_stepwise(self._h, S, _stream_ptr(stream)))

    def ks_run_traced(self, S: int, d_trace, stream=None):
        """d_trace: CUDA int32 tensor [M][S][2] (price after the step, Vmax)."""
        assert d_trace.is_cuda and d_trace.numel() >= self.M * S * 2
        _check(load().ks_run_traced(self._h, S, d_trace.data_ptr(), _stream_ptr(stream)))

    def ks_read_books(self, dst, stream=None):
        _check(load().ks_read_books(self._h, _ptr_of(dst), _stream_ptr(stream)))

    def ks_read_stats(self, dst, stream=None):
        _check(load().ks_read_stats(self._h, _ptr_of(dst), _stream_ptr(stream)))

    def ks_write_books(self, src, stream=None):
        _check(load().ks_write_books(self._h, _ptr_of(src), _stream_ptr(stream)))

    def ks_set_option(self, option: int, value: int):
        _check(load().ks_set_option(self._h, option, value))

    def ks_error_state(self):
        _check(load().ks_error_state(self._h))

    def ks_plan_string(self) -> str:
        buf = C.create_string_buffer(128)
        _check(load().ks_plan_string(self._h, buf, 128))
        return buf.value.decode()

    def ks_destroy(self):
        if self._h:
            load().ks_destroy(self._h)
            self._h = C.c_void_p(None)

    # -- conveniences for tests / bench (copies + a synchronize, nothing else) -----------------
    def books_to_host(self) -> np.ndarray:
        import torch
        out = torch.empty((self.M, 2, self.L), dtype=torch.int32, device="cpu").pin_memory()
        self.ks_read_books(out)
        torch.cuda.current_stream().synchronize()
        return out.numpy().copy()

    def stats_to_host(self) -> np.ndarray:
        import torch
        out = torch.empty((self.M, 16), dtype=torch.int64, device="cpu").pin_memory()
        self.ks_read_stats(out)
        torch.cuda.current_stream().synchronize()
        return out.numpy().copy()

    def __del__(self):
        try:
            self.ks_destroy()
        except Exception:
            pass


def ks_trace_stats(d_trace, M: int, S: int, K: int, d_out=None, stream=None):
    """d_trace: CUDA int32 [M][S][2]; returns (or fills) a CUDA float64 tensor [M][4 + 2K]."""
    import torch
    if d_out is None:
        d_out = torch.empty((M, 4 + 2 * K), dtype=torch.float64, device=d_trace.device)
    assert d_trace.is_cuda and d_out.is_cuda and d_out.numel() >= M * (4 + 2 * K)
    _check(load().ks_trace_stats(d_trace.data_ptr(), M, S, K, d_out.data_ptr(), _stream_ptr(stream)))
    return d_out


def ks_depth_bound_static(d_books, M: int, L: int, d_out, stream=None):
    """Largest per-side depth total of the book image d_books (CUDA int32 [M][2][L]) -> d_out (CUDA
    int64 tensor, one element, read it as uint64; all ones = a negative entry).  For callers that may
    not allocate device memory: the kernel's working memory is an array inside the library, so both
    tensors are the caller's and nothing is allocated here or in the library (include/kineticsim.h
    has the limit M <= KS_DEPTH_BOUND_STATIC_MAX_M and the rule that overlapping calls race)."""
    _check(load().ks_depth_bound_static(_ptr_of(d_books), M, L, _ptr_of(d_out), _stream_ptr(stream)))


def ks_bench_smem_atomic(mode, delta, L, threads=256, ctas_per_sm=8, iters=2000, warmup=2, reps=5, stream=None):
    ops, sec = C.c_double(0), C.c_double(0)
    _check(load_bench().ks_bench_smem_atomic(mode, delta, L, threads, ctas_per_sm, iters, warmup, reps,
                                       _stream_ptr(stream), C.byref(ops), C.byref(sec)))
    return ops.value, sec.value


def ks_bench_generate_only(params: dict, M, L, A, S, threads=256, warmup=1, reps=3, stream=None):
    ev, sec = C.c_double(0), C.c_double(0)
    P = _params(params)
    _check(load_bench().ks_bench_generate_only(C.byref(P), M, L, A, S, threads, warmup, reps, _stream_ptr(stream),
                                         C.byref(ev), C.byref(sec)))
    return ev.value, sec.value


def ks_bench_int_pipe(kind, threads=256, ctas_per_sm=8, iters=4000, warmup=2, reps=5, stream=None):
    ops, sec = C.c_double(0), C.c_double(0)
    _check(load_bench().ks_bench_int_pipe(kind, threads, ctas_per_sm, iters, warmup, reps, _stream_ptr(stream),
                                    C.byref(ops), C.byref(sec)))
    return ops.value, sec.value
