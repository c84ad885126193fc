// ks_device.cuh -- device side of the call-auction clearing library (sm_100a).
//
// One CTA per market.  The int32 book (bid[L], ask[L]) lives in shared memory for all S steps
// (Alg.1).  Per step: every thread generates orders for its agents with
// Philox4x32-10 and adds them to the book with shared-memory atomics (a1, a2); warp 0 then clears
// the ACTIVE WINDOW of the book with a register-blocked warp-shuffle scan (a3-a5) and updates the
// price state and the int64 statistics (a6).  Two __syncthreads() per step.
//
// Why a window is enough: let amin be the lowest tick with ask
// depth and bmax the highest tick with bid depth in the combined book.  V[p] = min(D[p], S[p]) is
// zero outside [amin, bmax], and for p < amin (p > bmax) the residual formula leaves bid[p]
// (ask[p]) untouched because D[p+1] >= Vmax (S[p-1] >= Vmax).  So scanning any tick range
// [lo, hi] with lo <= amin and hi >= bmax gives exactly the full-grid result of Eq.1-2.  New
// orders land within dmax ticks of `last`, and the resting book's bounds are tracked from the
// previous clearing, so the window is ~2*dmax+1 ticks wide instead of L.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace ks {

constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;
constexpr uint64_t kHashBasis = 0xcbf29ce484222325ull;
constexpr uint64_t kHashPrime = 0x100000001b3ull;

// record field indices (include/kineticsim.h, ks_market_stats)
enum { F_STEPS = 0, F_NTRADES, F_SUMVOL, F_SUMPX, F_SUMPX2, F_SUMPXVOL, F_SUMRET, F_SUMRET2,
       F_SUMRET3, F_SUMRET4, F_SUBBUY, F_SUBSELL, F_LAST, F_PREV, F_HASH, F_NORDERS };

struct KernelParams {
  int32_t* books;        // DEVICE [M][2][L]
  long long* recs;       // DEVICE [M][16]
  uint32_t k0[10];       // Philox round keys, word 0 (host-precomputed key schedule)
  uint32_t k1[10];       // word 1
  int32_t M, L, A;
  uint32_t market_base;
  int32_t noise_delta, noise_n, noise_qmax;      // noise_n = 2*delta+1
  int32_t maker_spread_max, maker_qty;
  int32_t mom_n, mom_qmax;                        // mom_n = mom_delta+1
  int32_t dmax;                                   // largest |tick - last| any rule can produce
  int32_t fresh;                                  // books are known to be all zero: skip the load
  int32_t force_generic;                          // ablation/test: always use the chunked scan
  long long S;                                    // steps to run
  long long orders_per_step;                      // A + number of makers
};

__device__ __forceinline__ uint32_t hi32(uint64_t x) { return (uint32_t)(x >> 32); }
__device__ __forceinline__ uint32_t lo32(uint64_t x) { return (uint32_t)x; }

// Values of the first two Philox rounds that do not depend on the agent.
// Round 0 on ctr = (a, t, m, 0):  n0 = hi(M1*m) ^ t ^ k0[0], n1 = lo(M1*m)      (uniform)
//                                 n2 = hi(M0*a) ^ k1[0],     n3 = lo(M0*a)      (per agent)
// Round 1 on (n0, n1, n2, n3):    d0 = hi(M1*n2) ^ n1 ^ k0[1], d1 = lo(M1*n2)   (per agent)
//                                 d2 = hi(M0*n0) ^ n3 ^ k1[1], d3 = lo(M0*n0)   (d3 uniform)
struct StepUniform {
  uint32_t n1k;   // n1 ^ k0[1]
  uint32_t d2x;   // hi(M0*n0) ^ k1[1]
  uint32_t d3;    // lo(M0*n0)
};

__device__ __forceinline__ StepUniform step_uniform(const KernelParams& P, uint32_t market, uint32_t t) {
  uint64_t pm = (uint64_t)kPhiloxM1 * market;
  uint32_t n0 = hi32(pm) ^ t ^ P.k0[0];
  uint64_t q0 = (uint64_t)kPhiloxM0 * n0;
  StepUniform u;
  u.n1k = lo32(pm) ^ P.k0[1];
  u.d2x = hi32(q0) ^ P.k1[1];
  u.d3 = lo32(q0);
  return u;
}

// Philox4x32-10 block of agent a; returns output words w0, w1, w2 (w3 is reserved, unused).
__device__ __forceinline__ void philox_agent(const KernelParams& P, const StepUniform& u, uint32_t a,
                                             uint32_t& w0, uint32_t& w1, uint32_t& w2) {
  uint64_t p0 = (uint64_t)kPhiloxM0 * a;
  uint32_t n2 = hi32(p0) ^ P.k1[0];
  uint32_t n3 = lo32(p0);
  uint64_t p1 = (uint64_t)kPhiloxM1 * n2;
  uint32_t c0 = hi32(p1) ^ u.n1k;
  uint32_t c1 = lo32(p1);
  uint32_t c2 = u.d2x ^ n3;
  uint32_t c3 = u.d3;
#pragma unroll
  for (int r = 2; r < 10; ++r) {
    uint64_t a0 = (uint64_t)kPhiloxM0 * c0;
    uint64_t a1 = (uint64_t)kPhiloxM1 * c2;
    uint32_t t0 = hi32(a1) ^ c1 ^ P.k0[r];
    uint32_t t2 = hi32(a0) ^ c3 ^ P.k1[r];
    c1 = lo32(a1);
    c3 = lo32(a0);
    c0 = t0;
    c2 = t2;
  }
  w0 = c0; w1 = c1; w2 = c2;
}

// a2: add one order to the shared-memory book.  ATOM 0: plain atomicAdd (ATOMS.ADD, result
// unused).  ATOM 1: warp-aggregated -- lanes with the same address elect a leader that adds the
// group's sum (north_star (3)); kept as an ablation switch.
template <int ATOM>
__device__ __forceinline__ void book_add(int32_t* book, int idx, int q, int& sink) {
  if (ATOM == 0) {
    atomicAdd(&book[idx], q);
  } else if (ATOM == 2) {
    sink ^= idx * 131 + q;               // microbenchmark only: no memory access (ks_bench_generate_only)
  } else {
    unsigned act = __activemask();
    unsigned peers = __match_any_sync(act, idx);
    int sum = __reduce_add_sync(peers, q);
    if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(&book[idx], sum);
  }
}

__device__ __forceinline__ int clamp_tick(int x, int L) { return min(max(x, 0), L - 1); }

// a1 noise rule.  CLAMP = false is the fast path used when last-delta >= 0 and last+delta <= L-1
// (a per-step uniform test), where the clamp is the identity.
template <int ATOM, bool CLAMP>
__device__ __forceinline__ void noise_order(const KernelParams& P, int32_t* book, int last,
                                            uint32_t w0, uint32_t w1, uint32_t w2, int& sink) {
  int o = (int)__umulhi(w1, (uint32_t)P.noise_n);
  int q = 1 + (int)__umulhi(w2, (uint32_t)P.noise_qmax);
  bool buy = (int32_t)w0 < 0;
  // buy: last - (o - delta) = (last + delta) - o ; sell: last + (o - delta) = (last - delta) + o
  int tick = buy ? (last + P.noise_delta) - o : (last - P.noise_delta) + o;
  if (CLAMP) tick = clamp_tick(tick, P.L);
  book_add<ATOM>(book, buy ? tick : tick + P.L, q, sink);
}

template <int ATOM, bool CLAMP>
__device__ __forceinline__ void generate_noise(const KernelParams& P, int32_t* book, const StepUniform& u,
                                               int last, uint32_t first, uint32_t a_end, uint32_t a_step,
                                               int& sink) {
  // agents first, first+a_step, ... < a_end
#pragma unroll 4
  for (uint32_t a = first; a < a_end; a += a_step) {
    uint32_t w0, w1, w2;
    philox_agent(P, u, a, w0, w1, w2);
    noise_order<ATOM, CLAMP>(P, book, last, w0, w1, w2, sink);
  }
}

// a1 maker rule: both sides, fixed quantity; only w1 is used.
template <int ATOM>
__device__ __forceinline__ void generate_maker(const KernelParams& P, int32_t* book, const StepUniform& u,
                                               int last, uint32_t first, uint32_t a_end, uint32_t a_step,
                                               int& sink) {
#pragma unroll 2
  for (uint32_t a = first; a < a_end; a += a_step) {
    uint32_t w0, w1, w2;
    philox_agent(P, u, a, w0, w1, w2);
    int s = 1 + (int)__umulhi(w1, (uint32_t)P.maker_spread_max);
    book_add<ATOM>(book, clamp_tick(last - s, P.L), P.maker_qty, sink);
    book_add<ATOM>(book, clamp_tick(last + s, P.L) + P.L, P.maker_qty, sink);
  }
}

// a1 momentum rule: dp = last - prev is uniform over the market-step.
template <int ATOM>
__device__ __forceinline__ void generate_momentum(const KernelParams& P, int32_t* book, const StepUniform& u,
                                                  int last, int dp, uint32_t first, uint32_t a_end,
                                                  uint32_t a_step, int& sink) {
#pragma unroll 2
  for (uint32_t a = first; a < a_end; a += a_step) {
    uint32_t w0, w1, w2;
    philox_agent(P, u, a, w0, w1, w2);
    bool buy = dp > 0 ? true : (dp < 0 ? false : ((int32_t)w0 < 0));
    int o = (int)__umulhi(w1, (uint32_t)P.mom_n);
    int q = 1 + (int)__umulhi(w2, (uint32_t)P.mom_qmax);
    int tick = clamp_tick(buy ? last + o : last - o, P.L);
    book_add<ATOM>(book, buy ? tick : tick + P.L, q, sink);
  }
}

// a1 + a2 for one market-step: every thread of the CTA generates the orders of its agents.
// MODEL 1: agent a = 3j + c has type c; each class runs in its own warp-uniform loop (integer
// atomics commute, so the agent -> thread mapping cannot change a byte of the result).
template <int MODEL, int ATOM>
__device__ __forceinline__ void generate_step(const KernelParams& P, int32_t* book, const StepUniform& u,
                                              int last, int prev, int tid, int T, int& sink) {
  const uint32_t A = (uint32_t)P.A;
  const bool noclamp = (last - P.noise_delta >= 0) && (last + P.noise_delta <= P.L - 1);
  if (MODEL == 0) {
    if (noclamp) generate_noise<ATOM, false>(P, book, u, last, (uint32_t)tid, A, (uint32_t)T, sink);
    else         generate_noise<ATOM, true >(P, book, u, last, (uint32_t)tid, A, (uint32_t)T, sink);
  } else {
    const uint32_t st = 3u * (uint32_t)T;
    if (noclamp) generate_noise<ATOM, false>(P, book, u, last, 3u * tid, A, st, sink);
    else         generate_noise<ATOM, true >(P, book, u, last, 3u * tid, A, st, sink);
    generate_maker<ATOM>(P, book, u, last, 3u * tid + 1u, A, st, sink);
    generate_momentum<ATOM>(P, book, u, last, last - prev, 3u * tid + 2u, A, st, sink);
  }
}

// ---------------------------------------------------------------------------------------------
// a3-a5, one warp, window of at most 32*K ticks starting at `base` (a multiple of K).
// Lane i owns ticks base + i*K .. base + i*K + K-1 in registers.
//   D[p] = (bids of higher lanes) + (own bids at ticks >= p)      Eq.1, suffix
//   S[p] = (asks of lower lanes)  + (own asks at ticks <= p)      Eq.1, prefix
//   V = min(D, S); Vmax by REDUX max; p* = lowest tick attaining it
//   residual: bid <- min(bid, max(0, D - Vmax)), ask <- min(ask, max(0, S - Vmax))
// Also returns conservative bounds of the residual book inside the window (bmax: highest tick
// with bid depth, else base-1; amin: lowest tick with ask depth, else base+32K).
// ---------------------------------------------------------------------------------------------
template <int K>
__device__ __forceinline__ void clear_window(int32_t* book, int L, int base, int lane,
                                             int& vmax, int& pstar, int& bmax_new, int& amin_new) {
  static_assert(K % 4 == 0, "K must be a multiple of 4 (16-byte shared-memory vectors)");
  const unsigned FULL = 0xffffffffu;
  const int tick0 = base + lane * K;
  const bool in = tick0 < L;            // L and base are multiples of K: a lane is all in or all out
  int b[K], a[K];
#pragma unroll
  for (int v = 0; v < K / 4; ++v) {
    int4 vb = make_int4(0, 0, 0, 0), va = make_int4(0, 0, 0, 0);
    if (in) {
      vb = *reinterpret_cast<const int4*>(book + tick0 + 4 * v);
      va = *reinterpret_cast<const int4*>(book + L + tick0 + 4 * v);
    }
    b[4 * v] = vb.x; b[4 * v + 1] = vb.y; b[4 * v + 2] = vb.z; b[4 * v + 3] = vb.w;
    a[4 * v] = va.x; a[4 * v + 1] = va.y; a[4 * v + 2] = va.z; a[4 * v + 3] = va.w;
  }
  int tb = 0, ta = 0;
#pragma unroll
  for (int j = 0; j < K; ++j) { tb += b[j]; ta += a[j]; }
  int sufb = tb, prea = ta;             // inclusive suffix of bids / prefix of asks over lanes
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    int vb = __shfl_down_sync(FULL, sufb, d);
    int va = __shfl_up_sync(FULL, prea, d);
    if (lane + d < 32) sufb += vb;
    if (lane >= d) prea += va;
  }
  // profiles are recomputed in the residual pass instead of being kept: K fewer registers x 2
  const int D0 = sufb, S0 = prea - ta;
  int bestV = 0, bestp = 0x7fffffff;
  {
    int Drun = D0, Srun = S0;
#pragma unroll
    for (int j = 0; j < K; ++j) {
      Srun += a[j];
      int V = min(Drun, Srun);                          // D[p], S[p] at p = tick0 + j
      Drun -= b[j];
      if (V > bestV) { bestV = V; bestp = tick0 + j; }  // strict >: lowest tick within the lane
    }
  }
  vmax = __reduce_max_sync(FULL, bestV);
  pstar = __reduce_min_sync(FULL, bestV == vmax ? bestp : 0x7fffffff);
  int lb = -1, la = 0x7fffffff;
  if (vmax > 0) {
    int Drun = D0 - vmax, Srun = S0 - vmax;
#pragma unroll
    for (int j = 0; j < K; ++j) {
      Srun += a[j];
      int nbid = min(b[j], max(0, Drun));
      Drun -= b[j];
      b[j] = nbid;
      a[j] = min(a[j], max(0, Srun));
    }
    if (in) {
#pragma unroll
      for (int v = 0; v < K / 4; ++v) {
        *reinterpret_cast<int4*>(book + tick0 + 4 * v) = make_int4(b[4 * v], b[4 * v + 1], b[4 * v + 2], b[4 * v + 3]);
        *reinterpret_cast<int4*>(book + L + tick0 + 4 * v) = make_int4(a[4 * v], a[4 * v + 1], a[4 * v + 2], a[4 * v + 3]);
      }
    }
  }
#pragma unroll
  for (int j = 0; j < K; ++j) {
    if (b[j] > 0) lb = tick0 + j;                      // ascending: the highest wins
    if (a[K - 1 - j] > 0) la = tick0 + K - 1 - j;      // descending: the lowest wins
  }
  bmax_new = __reduce_max_sync(FULL, lb);
  amin_new = __reduce_min_sync(FULL, la);
  if (bmax_new < 0) bmax_new = base - 1;
  if (amin_new == 0x7fffffff) amin_new = min(L, base + 32 * K);
}

// General window of any width: chunks of 128 ticks, three passes (total bid depth; profiles and
// arg max; residual and bounds).  Slow path: first step after a ks_write_books, or a window wider
// than 256 ticks.  Same definitions as clear_window.
static __device__ __noinline__ void clear_generic(int32_t* book, int L, int base, int top, int lane,
                                           int& vmax, int& pstar, int& bmax_new, int& amin_new) {
  const unsigned FULL = 0xffffffffu;
  // pass 0: total bid depth of the window
  int tbsum = 0;
  for (int c = base; c <= top; c += 128) {
    int t = c + lane * 4;
    if (t < L) { int4 vb = *reinterpret_cast<const int4*>(book + t); tbsum += vb.x + vb.y + vb.z + vb.w; }
  }
  const int TB = __reduce_add_sync(FULL, tbsum);
  int bestV = 0, bestp = 0x7fffffff;
  int lb = -1, la = 0x7fffffff;
  vmax = 0; pstar = 0x7fffffff;
  for (int pass = 1; pass <= 2; ++pass) {
    int carryB = 0, carryA = 0;   // bid depth strictly below the chunk / ask depth strictly below
    for (int c = base; c <= top; c += 128) {
      int t = c + lane * 4;
      bool in = t < L;
      int4 vb = make_int4(0, 0, 0, 0), va = vb;
      if (in) { vb = *reinterpret_cast<const int4*>(book + t); va = *reinterpret_cast<const int4*>(book + L + t); }
      int b[4] = {vb.x, vb.y, vb.z, vb.w}, a[4] = {va.x, va.y, va.z, va.w};
      int tb = b[0] + b[1] + b[2] + b[3], ta = a[0] + a[1] + a[2] + a[3];
      int preb = tb, prea = ta;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) {
        int xb = __shfl_up_sync(FULL, preb, d);
        int xa = __shfl_up_sync(FULL, prea, d);
        if (lane >= d) { preb += xb; prea += xa; }
      }
      int below = carryB + preb - tb;         // bid depth at ticks < t
      int Srun = carryA + prea - ta;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        int D = TB - below;                   // bids at ticks >= t+j
        Srun += a[j];
        below += b[j];
        if (pass == 1) {
          int V = min(D, Srun);
          if (V > bestV) { bestV = V; bestp = t + j; }
        } else {
          b[j] = min(b[j], max(0, D - vmax));
          a[j] = min(a[j], max(0, Srun - vmax));
          if (b[j] > 0) lb = max(lb, t + j);
          if (a[j] > 0) la = min(la, t + j);
        }
      }
      if (pass == 2 && in && vmax > 0) {
        *reinterpret_cast<int4*>(book + t) = make_int4(b[0], b[1], b[2], b[3]);
        *reinterpret_cast<int4*>(book + L + t) = make_int4(a[0], a[1], a[2], a[3]);
      }
      carryB += __shfl_sync(FULL, preb, 31);
      carryA += __shfl_sync(FULL, prea, 31);
    }
    if (pass == 1) {
      vmax = __reduce_max_sync(FULL, bestV);
      pstar = __reduce_min_sync(FULL, bestV == vmax ? bestp : 0x7fffffff);
    }
  }
  bmax_new = __reduce_max_sync(FULL, lb);
  amin_new = __reduce_min_sync(FULL, la);
  if (bmax_new < 0) bmax_new = base - 1;
  if (amin_new == 0x7fffffff) amin_new = min(L, top + 1);
}

}  // namespace ks
