/*
 * kineticsim.h -- C ABI of the B200-native (sm_100a) call-auction clearing library.
 *
 * The library runs the hot path of KineticSim (arxiv/paper_2606_21784; citations are PAPER.md
 * line numbers): M independent limit-order-book markets, each with L price ticks and A agents,
 * advanced S steps by ONE launch of a persistent kernel that keeps every market's book in shared
 * memory for all S steps (Alg.1; SIII-A/B) and touches HBM
 * once to load and once to store the state (Eq.6).  Per step and market:
 *   1. every agent a draws one Philox4x32-10 block keyed by (seed, market, step, agent) and turns
 *      it into a limit order (side, tick, integer quantity)       (SIII-C)
 *   2. orders are added to the int32 bid/ask depth per tick with shared-memory atomics
 *                                                          (Alg.1 l.10-13)
 *   3. D[p] = sum_{q>=p} bid[q], S[p] = sum_{q<=p} ask[q]              (Eq.1)
 *   4. p* = lowest p maximising V[p] = min(D[p], S[p]), Vmax = V[p*]   (Eq.2; ties
 *      to the lowest tick)
 *   5. price-priority allocation; the unfilled remainder rests for the next step:
 *      bid[p] <- min(bid[p], max(0, D[p]-Vmax)), ask[p] <- min(ask[p], max(0, S[p]-Vmax));
 *      nothing changes when Vmax = 0            (SIV-C)
 *   6. prev <- last; last <- p* if Vmax > 0; int64 statistics accumulate
 *
 * Conventions.  No C++ types, exceptions or torch types cross this boundary.  Every pointer
 * argument says whether it is a HOST or a DEVICE pointer.  `stream` is a cudaStream_t passed as
 * void* (NULL = the legacy default stream).  Unless stated otherwise a call only ENQUEUES work on
 * `stream` and returns; the caller synchronises, and calls on one ks_sim must be stream-ordered
 * by the caller.  On an error return nothing has been enqueued.  There is no CPU fallback: with
 * no CUDA device every call that needs one returns KS_ERR_CUDA.
 */
#ifndef KINETICSIM_H_
#define KINETICSIM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define KS_API __attribute__((visibility("default")))
#else
#define KS_API
#endif

typedef struct ks_sim ks_sim; /* opaque host-side handle, owned by the library */

typedef enum {
  KS_OK = 0,
  KS_ERR_INVALID_ARG = -1, /* NULL pointer, M < 1, A < 0, S < 0, L not a power of two or < 32, bad params */
  KS_ERR_UNSUPPORTED = -2, /* L > 32768 (p* must fit the 16-bit field of the trajectory hash), or a book
                              that does not fit this device's shared memory.  16384 < L <= 32768 runs on a
                              thread-block cluster (DSMEM), see KS_OPT_CLUSTER_SIZE                        */
  KS_ERR_OVERFLOW = -3,    /* a per-side depth sum could leave int32 (refused before the run), or a
                              statistic DID leave int64 during an earlier run (sticky, see ks_run)        */
  KS_ERR_CUDA = -4,        /* a CUDA call failed; text in ks_last_error()                                 */
  KS_ERR_NOMEM = -5        /* host allocation failed                                                      */
} ks_status;

typedef enum {
  KS_MODEL_ZI = 0,  /* every agent is a zero-intelligence noise trader (BASELINE.json configs[0..3]) */
  KS_MODEL_MIX3 = 1, /* agent a: a%3 = 0 noise, 1 market maker, 2 momentum (BASELINE.json configs[4]) */
  /* The same rules under the PACKED4 draw contract (reading A22) -- a
   * separately named contract with its own orders, NOT the BASELINE.json one: one Philox block
   * serves four consecutive agents, w = Philox(ctr = (a >> 2, step, market, 0), key)[a & 3], and
   * every draw comes out of that word by successive multiply-extract: o = mulhi(w, n),
   * x1 = lo32(w*n); q = 1 + mulhi(x1, qmax), x2 = lo32(x1*qmax); coin = x2 >> 31 (maker:
   * s = 1 + mulhi(w, spread_max)).  Plain atomics only (KS_OPT_ATOMIC_MODE 0). */
  KS_MODEL_ZI_PACKED4 = 2,
  KS_MODEL_MIX3_PACKED4 = 3,
  /* The paper's own agent model (SIII-C; reading A24),
   * a separately named model beside the BASELINE.json ones.  Reference price: the mid of the RESTING
   * book at the start of the step in doubled-integer form, mid2 = bb + ba (highest bid tick + lowest
   * ask tick), or 2*last when a side is empty (Eq.3); round(m2/2) = floor((m2+1)/2).
   * Classes are contiguous index ranges: agents [0, A - paper_n_mom - paper_n_maker) noise, then
   * paper_n_mom momentum, then paper_n_maker makers.  Words of Philox(ctr = (a, step, market, 0)):
   *   noise     buy = w0>>31; eta = mulhi(w1, 2*noise_delta+1) - noise_delta; p = round(mid + eta);
   *             q = 1 + mulhi(w2, noise_qmax)
   *   momentum  buy = sgn(mid2 - previous mid2) > 0, < 0 -> sell, = 0 -> w0>>31; p = round(mid +/- 1);
   *             q = 1 + mulhi(w2, mom_qmax)
   *   maker     buys iff (a + step) is even; p = round(mid - h) for a bid, round(mid + h) for an ask,
   *             h = maker_spread_max; q = 1 + mulhi(w2, maker_qty); never marketable
   *   noise and momentum orders are marketable iff (w3 >> 16) < paper_pmkt_q16: p = L-1 for a buy,
   *   0 for a sell.  p is clamped to the grid.  Record field f[13] holds mid2 of the last executed
   *   step (2*init before the first) instead of the previous price.
   * L <= 16384 (no cluster path), plain atomics only. */
  KS_MODEL_PAPER = 4
} ks_model;

/*
 * Agent rules (SIII-C, in the integer form BASELINE.json fixes).  With
 * w0..w3 = Philox4x32-10(ctr = (agent, step, market, 0), key = (seed lo, seed hi)),
 * mulhi(w, n) = (uint64(w) * n) >> 32, clamp(x) = min(max(x, 0), L-1), and last / prev the last
 * two clearing prices as they were at the START of the step:
 *   noise     buy = w0 >> 31; o = mulhi(w1, 2*noise_delta+1) - noise_delta; q = 1 + mulhi(w2, noise_qmax)
 *             tick = buy ? clamp(last - o) : clamp(last + o)
 *   maker     s = 1 + mulhi(w1, maker_spread_max); bid maker_qty @ clamp(last - s) AND ask
 *             maker_qty @ clamp(last + s) (one agent event, two orders)
 *   momentum  dp = last - prev; buy = dp > 0 ? 1 : dp < 0 ? 0 : w0 >> 31; o = mulhi(w1, mom_delta+1)
 *             q = 1 + mulhi(w2, mom_qmax); tick = buy ? clamp(last + o) : clamp(last - o)
 * Ranges: 0 <= noise_delta, mom_delta, maker_spread_max-1 < L; 1 <= qmax, qty <= 2^20.
 */
typedef struct {
  int32_t model;            /* ks_model                                             */
  int32_t noise_delta;      /* noise offset uniform in [-noise_delta, +noise_delta] */
  int32_t noise_qmax;       /* noise quantity uniform in 1..noise_qmax              */
  int32_t maker_spread_max; /* maker spread uniform in 1..maker_spread_max          */
  int32_t maker_qty;        /* maker quantity posted on each side                   */
  int32_t mom_delta;        /* momentum offset uniform in [0, mom_delta]            */
  int32_t mom_qmax;         /* momentum quantity uniform in 1..mom_qmax             */
  int32_t init_price;       /* opening last = prev; < 0 means L/2                   */
  /* KS_MODEL_PAPER only (ignored otherwise; set to 0) */
  int32_t paper_n_mom;      /* number of momentum agents                            */
  int32_t paper_n_maker;    /* number of market makers                              */
  int32_t paper_pmkt_q16;   /* P_mkt = paper_pmkt_q16 / 65536, 0..65536             */
} ks_agent_params;

/*
 * Per-market statistics record, 128 bytes, integer sums only ("clearing statistics",
 * PAPER.md:302).  r = last_after - last_before of a step (0 on a no-trade step).
 *   f[0] steps       f[1] n_trades (steps with Vmax > 0)   f[2] sum Vmax       f[3] sum p*
 *   f[4] sum p*^2    f[5] sum p* * Vmax                    f[6] sum r          f[7] sum r^2
 *   f[8] sum r^3     f[9] sum r^4      f[10] submitted bid quantity   f[11] submitted ask quantity
 *   f[12] last       f[13] prev        f[14] trajectory hash (uint64) f[15] number of orders
 * Trajectory hash: h0 = 0xcbf29ce484222325; per step x = Vmax > 0 ? (uint64(Vmax) << 16 | p*) :
 * 0xFFFF; h = (h ^ x) * 0x100000001b3 mod 2^64 -- it pins every step's (p*, Vmax).
 */
typedef struct { int64_t f[16]; } ks_market_stats;

/* fp64 statistics derived on the HOST from one record by ks_derive_stats:
 *   d[0] mean clearing price = f3/f1        d[1] VWAP = f5/f2          d[2] volume per step = f2/f0
 *   d[3] mean return mu = f6/f0             d[4] return variance = f7/f0 - mu^2
 *   d[5] excess kurtosis = m4/var^2 - 3, m4 = (f9 - 4 mu f8 + 6 mu^2 f7)/f0 - 3 mu^4
 * A quantity with a zero denominator is NaN. */
typedef struct { double d[6]; } ks_derived_stats;

/* Bytes of the caller-owned DEVICE state buffer: int32 books[M][2][L] (side 0 = bid, 1 = ask),
 * then ks_market_stats rec[M], then 256 bytes of library scratch.  = M*(8*L+128) + 256.
 * Returns 0 for arguments ks_create would reject. */
KS_API size_t ks_state_bytes(int32_t M, int32_t L);

/*
 * Create a simulation of M markets x L ticks x A agents (Alg.1 "Require").
 *   out      HOST: receives the handle (freed by ks_destroy).
 *   p        HOST: agent parameters, copied.
 *   seed     Philox key.
 *   d_state  DEVICE: caller-owned buffer of ks_state_bytes(M, L) bytes, 16-byte aligned, on the
 *            CURRENT device (the handle remembers that device and makes it current inside every
 *            later call); the library never allocates or frees device memory and never frees
 *            d_state.  It IS the checkpoint: books, prices, step counter and accumulators live
 *            there between calls, and ks_attach resumes from a saved copy of it.
 * Enqueues the initialisation on `stream`: empty books, last = prev = init price, zero sums
 * (Alg.1 l.2-3; opening quotes per BASELINE.json: empty book, price L/2).
 * ks_create_ex additionally takes the global id of this shard's first market: Philox is keyed by
 * market_base + local index, so a market's trajectory does not depend on how the market range is
 * partitioned across GPUs.  ks_create(...) == ks_create_ex(..., market_base = 0, ...).
 */
KS_API ks_status ks_create(ks_sim** out, int32_t M, int32_t L, int32_t A, const ks_agent_params* p,
                           uint64_t seed, void* d_state, void* stream);
KS_API ks_status ks_create_ex(ks_sim** out, int32_t M, int32_t L, int32_t A, const ks_agent_params* p,
                              uint64_t seed, uint32_t market_base, void* d_state, void* stream);

/*
 * Resume from a checkpoint (the "final order book and clearing statistics in global memory" of
 * Alg.1 "Ensure", fed back in): a new handle over a d_state that ALREADY holds the
 * bytes an earlier handle left there (same M, L; the caller passes the same A, parameters, seed
 * and market_base to continue the same trajectory).  Nothing is initialised: books, prices, step
 * counter, sums and hash are taken as they are, so
 *     ks_run(S1) -> save d_state -> ... -> restore -> ks_attach -> ks_run(S2)
 * leaves the bytes of one uninterrupted ks_run(S1+S2).  Unlike the other calls this one
 * SYNCHRONISES `stream`: it reads the step counter and the largest per-side depth back from the
 * device for the overflow guards of ks_run.  Arguments and errors as ks_create_ex, plus
 * KS_ERR_INVALID_ARG when d_state holds a negative depth, or a record this library cannot have
 * written: EVERY market's record is checked on the device (step counter f[0] >= 0, last price f[12]
 * on the grid, f[13] on the grid -- or a valid doubled mid for KS_MODEL_PAPER); the guards of ks_run
 * continue from the LARGEST step counter found.
 */
KS_API ks_status ks_attach(ks_sim** out, int32_t M, int32_t L, int32_t A, const ks_agent_params* p,
                           uint64_t seed, uint32_t market_base, void* d_state, void* stream);

/*
 * Advance every market by S steps with ONE launch of the persistent kernel,
 * continuing from the state in d_state: the Philox step index is steps_done + i, so
 * ks_run(S1); ks_run(S2) leaves the same bytes as ks_run(S1+S2).  S = 0 is a no-op.
 * KS_ERR_OVERFLOW (nothing enqueued) when (steps_done+S) x per-step per-side inflow bound, plus
 * the depth injected by ks_write_books, could reach 2^31 (int32 book), or steps_done+S >= 2^32 - 8
 * (the kernels count steps in 32 bits and look up to 8 steps ahead).
 * Deferred errors.  (1) If the depth check of a preceding ks_write_books has not finished yet, the
 * host does NOT wait for it: the launch is ordered after the check on the device (an event wait on
 * `stream`, so `stream` may differ from the one ks_write_books used), the kernel reads the check's
 * result there and, when the bound
 * is violated (or a negative depth was stored), the whole launch returns without changing a byte
 * of d_state.  (2) The int64 sums of r^3 and r^4 (f[8], f[9]) can only overflow on wide grids
 * after very large price moves ((L-1)^4 x steps >= 2^63 at the earliest); the kernel detects the
 * signed overflow exactly when it happens.  Either event sets a sticky flag that the kernel writes
 * into host memory: every later ks_run* / ks_read_* / ks_write_books on this handle -- in
 * particular the first ks_read_* after the caller has synchronised the stream -- returns
 * KS_ERR_OVERFLOW (KS_ERR_INVALID_ARG for the negative depth), and the handle must be destroyed.
 */
KS_API ks_status ks_run(ks_sim* s, int64_t S, void* stream);

/*
 * ks_run that also records the per-step trace of this call (the paper "records
 * the price returns" of every market for its SIV-J sweep).
 *   d_trace  DEVICE, caller-owned, 8-byte aligned: int32 [M][S][2]; entry [m][i] = (price after
 *            step i of this call -- p* if the step traded, else the unchanged last price --,
 *            executed volume Vmax, 0 if none).  Written in 256-byte coalesced chunks, 8*M*S bytes
 *            in all; nothing else about the run changes (same bytes in d_state as ks_run).
 * Errors as ks_run, plus KS_ERR_INVALID_ARG for a NULL or misaligned d_trace.
 */
KS_API ks_status ks_run_traced(ks_sim* s, int64_t S, int32_t* d_trace, void* stream);

/*
 * Return statistics of a trace (SIV-J, Fig.7; reading A23), one kernel,
 * one warp per market.  d_trace: DEVICE int32 [M][S][2] as written by ks_run_traced.  d_out: DEVICE
 * double [M][4 + 2K].  With r_t = p_t - p_{t-1} between consecutive traced steps (n = S-1 returns):
 *   [0] volatility = population std of r       [1] excess kurtosis = m4/m2^2 - 3 (central moments)
 *   [2] volume per step = sum Vmax / S         [3] mean return
 *   [4 .. 4+K)    ACF_r(k),   k = 1..K:  sum_{t>k} (r_t - rbar)(r_{t-k} - rbar) / sum_t (r_t - rbar)^2
 *   [4+K .. 4+2K) ACF_|r|(k), k = 1..K
 * A quantity with a zero denominator is NaN.  Sums are exact integers (128-bit where needed); only
 * the final quotients are rounded.  Range: every |r_t| <= 46340 (L <= 32768 guarantees it) and
 * S^4 * max|r|^4 < 2^126.
 * KS_ERR_INVALID_ARG for NULL pointers, M < 1, S < 1, K < 0 or K > 256.
 */
KS_API ks_status ks_trace_stats(const int32_t* d_trace, int32_t M, int64_t S, int32_t K, double* d_out,
                                void* stream);

/* HOST-only, never blocks: KS_OK, or the sticky deferred error of this handle (see ks_run).  A
 * caller that has synchronised the stream after a run learns here whether that run was refused on
 * the device or overflowed a statistic. */
KS_API ks_status ks_error_state(ks_sim* s);

/* Copy the books / the records out of d_state.  dst: HOST or DEVICE pointer (cudaMemcpyDefault),
 * int32 [M][2][L] resp. ks_market_stats [M]; a host destination must stay valid until the stream
 * work is done (pinned memory makes the copy asynchronous).  Alg.1 "Ensure". */
KS_API ks_status ks_read_books(ks_sim* s, int32_t* dst, void* stream);
KS_API ks_status ks_read_stats(ks_sim* s, ks_market_stats* dst, void* stream);

/* Replace the resting books (test hook: "seeds the opening quotes").  src: HOST or
 * DEVICE pointer, int32 [M][2][L], every entry >= 0.  Records are left as they are.  Also enqueues
 * a depth check (one small kernel) whose result the next ks_run uses -- on the host if it has
 * finished by then, else on the device (see ks_run, deferred errors). */
KS_API ks_status ks_write_books(ks_sim* s, const int32_t* src, void* stream);

/*
 * Depth check of a book image for callers that have no device memory to lend and may not get any.
 *
 * What it computes is what the depth check behind ks_write_books / ks_attach computes: over all M
 * markets and both sides, the largest per-side depth total sum_p book[m][side][p] -- the number the
 * int32 overflow guard of ks_run needs (Eq.1: D and S are running sums of these entries
 * and must stay below 2^31) -- or 0xFFFFFFFFFFFFFFFF when any entry is negative.
 *
 * Who needs it.  Everywhere else in this library the kernels' working memory comes from the caller:
 * the depth check borrows a word from the 256-byte tail of d_state.  A caller who wants to vet an
 * image BEFORE a ks_sim exists -- a checkpoint about to go to ks_attach, books about to go to
 * ks_write_books -- has no d_state to lend, and often cannot make one: (1) a thread beside a running
 * simulation must not call cudaMalloc / cudaFree, because both wait for the whole device, i.e. for a
 * ks_run launch that holds the GPU for hundreds of milliseconds; (2) in a process whose framework has
 * already claimed all of HBM for its own pool, a raw cudaMalloc simply fails; (3) code under a
 * "no allocation after start-up" rule (a real-time loop, a plug-in whose host forbids it) may not ask.
 * For them the working memory of this one call lives INSIDE the library: a file-scope device array of
 * 32 + 2*KS_DEPTH_BOUND_STATIC_MAX_M 8-byte words (1 MiB + 256 B) that every GPU holds from the moment
 * it loads the library until the process exits, whether or not this call is ever made.
 *
 *   d_books  DEVICE, on the CURRENT device, 4-byte aligned: int32 [M][2][L] (the layout of
 *            ks_read_books); read only.
 *   M, L     as ks_create (L a power of two, 32..32768); M <= KS_DEPTH_BOUND_STATIC_MAX_M.
 *   d_out    DEVICE, on the current device, 8-byte aligned: receives the one 64-bit result.
 * Enqueues a 8-byte clear and ONE kernel on `stream` and returns; it calls no cudaMalloc, cudaFree,
 * cudaHostAlloc or any other allocating routine, and needs no ks_sim.
 * Errors (nothing enqueued): KS_ERR_INVALID_ARG for a NULL / misaligned pointer or a bad M / L;
 * KS_ERR_UNSUPPORTED, with the limit in ks_last_error(), when M > KS_DEPTH_BOUND_STATIC_MAX_M -- use
 * ks_write_books / ks_attach on a real d_state for larger images, or check the image in slices of
 * markets and take the maximum; KS_ERR_CUDA when a CUDA call fails.
 *
 * First call on each device.  The library looks up the device address of its array once per device
 * (cudaGetSymbolAddress, with that device current) and remembers it.  That look-up makes the CUDA
 * runtime load this library's device code on that GPU if it has not yet done so, so make the first
 * call on every device during start-up, before any stream capture is begun.
 *
 * One array, shared by everybody.  All calls on a device -- from any thread, on any stream -- use the
 * same words, and the array keeps whatever the previous call left in it.  The call clears the one word
 * that has to start at zero (a ticket counter) itself, on `stream`, and every other word it reads has
 * been written earlier in the same call, so back-to-back calls on ONE stream are safe.  Two calls that
 * can overlap on the GPU (different streams with no ordering between them, or two host threads each
 * on their own stream) race on those words and may both return garbage: order them yourself.
 */
#define KS_DEPTH_BOUND_STATIC_MAX_M 65536
KS_API ks_status ks_depth_bound_static(const int32_t* d_books, int32_t M, int32_t L, uint64_t* d_out,
                                       void* stream);

/* Tuning / ablation switches; none of them changes a single output byte.  Returns
 * KS_ERR_INVALID_ARG for an unknown option or value. */
typedef enum {
  KS_OPT_BLOCK_THREADS = 0, /* threads per CTA: 0 = automatic, else 32..1024, multiple of 32          */
  KS_OPT_ATOMIC_MODE = 1,   /* 0 = plain shared-memory atomicAdd, 1 = warp-aggregated (__match_any_sync) */
  KS_OPT_CLEAR_PATH = 2,    /* 0 = automatic (windowed one-warp scan), 1 = force the chunked general scan */
  KS_OPT_PIPELINE = 4,      /* the decoupled kernel (generating warps fill a ring of price-independent relative order
                               histograms up to KS_OPT_RING_DEPTH steps ahead; the LAST warp of the CTA is the market's
                               clearing warp, holds no agents, merges them at the step's price and clears):
                               0 = automatic (when the grid underfills the GPU, i.e. step latency is what counts, or
                               when an SM holds only a few markets, M <= 16 x #SMs; and always as part of the
                               automatic two-steps-per-pass plan, see KS_OPT_STEP_PAIRS), 1 = never, 2 = whenever
                               legal.  Legal for KS_MODEL_ZI / KS_MODEL_ZI_PACKED4 with plain atomics, >= 64 threads,
                               L <= 16384 and book + histogram ring fitting shared memory; and for KS_MODEL_MIX3
                               (literal draws) in its two-steps-per-pass form only: plain atomics, maker_spread_max
                               <= 64, mom_delta < 64, 64 <= threads <= 160, KS_OPT_REL_COLUMNS 0, KS_OPT_RING_DEPTH 0 */
  KS_OPT_REL_COLUMNS = 5,   /* decoupled kernel only: 0 = one int32 per histogram bin, 1 = 32 lane columns per
                               bin (column = lane = bank: a warp's atomics never conflict) -- the
                               aggregation ablation of north_star (3); two-deep ring, one step per pass         */
  KS_OPT_RING_DEPTH = 6,    /* decoupled kernel only: how many steps the generating warps may run ahead of the
                               clearing warp = number of relative histograms in the ring: 0 = automatic (4 when the
                               step latency counts, M <= 2 x #SMs; 2 when throughput does, M > 2 x #SMs, or with
                               KS_OPT_REL_COLUMNS; always 4 under two steps per pass), 2 or 4 = forced (a forced
                               value rules out two steps per pass)                                            */
  KS_OPT_STEP_PAIRS = 7,    /* decoupled kernel, 64..160 threads: the generating warps make TWO steps per pass over
                               their agents (the step-independent Philox rounds and the counter add are shared: 18
                               multiplies per event instead of 19) and hand them over together (ring of 4, the
                               clearing warp keeps the record).  KS_MODEL_ZI (literal draws), and KS_MODEL_MIX3 with
                               maker_spread_max <= 64 and mom_delta < 64 (every rule binned relative to the step's
                               opening price and price change).  0 = automatic (ZI: >= 4 events per generating
                               thread, i.e. A >= 1024, or A >= 512 when M <= 16 x #SMs; MIX3: A >= 1536 and four CTAs
                               fitting an SM; the grid not underfilled; no forced block size), 1 = never,
                               2 = whenever legal                                                              */
  KS_OPT_CLUSTER_SIZE = 3   /* CTAs per market: 0 = automatic (1 while the book fits one CTA's shared memory,
                               i.e. L <= 16384; else L/16384), 1, or 2/4/8 = thread-block cluster with the
                               book split across the CTAs' shared memory (DSMEM); needs L/value >= 32 and
                               KS_OPT_ATOMIC_MODE 0                                                          */
} ks_option;
KS_API ks_status ks_set_option(ks_sim* s, int32_t option, int32_t value);

/* HOST-only: which kernel and launch shape the next ks_run on this handle will use under its current
 * options, as text ("ks_persistent_kernel T=32", "ks_decoupled_kernel T=96 ring=4 steps_per_pass=2",
 * "ks_cluster_kernel C=2") -- for logs and for bench.py, which must know how many multiplies per
 * event the chosen kernel executes.  buf: HOST, n bytes, always NUL-terminated. */
KS_API ks_status ks_plan_string(ks_sim* s, char* buf, size_t n);

/* HOST-only helper: derive the fp64 statistics of n records. */
KS_API void ks_derive_stats(const ks_market_stats* rec, ks_derived_stats* out, int64_t n);

KS_API void ks_destroy(ks_sim* s);

/* Text of the last error on this thread; never NULL. */
KS_API const char* ks_last_error(void);

/* Number of kernels this library has launched in this process (all handles). */
KS_API int64_t ks_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* KINETICSIM_H_ */
