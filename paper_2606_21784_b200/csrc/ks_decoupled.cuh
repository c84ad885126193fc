// ks_decoupled.cuh -- the latency kernel: order generation DECOUPLED from the clearing price.
//
// In ks_persistent_kernel a step is a chain: generate (needs the price) | barrier | clear (gives
// the next price) | barrier.  When many markets share an SM they hide each other's chains (C4);
// when the grid underfills the GPU (C3: 32 markets, C1: one) the chain IS the run time.  But for a
// zero-intelligence agent only the TICK depends on the price, not the order: offset draw o, side
// and quantity are pure functions of (seed, market, step, agent).  So here the generating warps
// never see a price.  They add their orders to a relative histogram (sell[o], buy[n-1-o]: bin i of
// either side means tick last - delta + i; ATOM 4 / 5 of ks_device.cuh), double-buffered by step
// parity, and run up to two steps ahead; ONE clearing warp per market (which holds no agents) takes
// buffer (s & 1) at the current price -- exactly the rule's ticks, clamped to the grid -- zeroes it,
// hands it back, and clears (a3-a6).  In the common case (no order clamped, window <= 128 ticks)
// the histogram is not even merged into the book first: each lane adds its ticks' bins to the
// depth it loads for the scan.  The per-step critical path is max(generate, clear) with no price
// round trip between the two, and the SM's other warps never idle at a barrier.
//
// Synchronisation: four named barriers, full[b] (generating warps arrive, clearing warp waits)
// and free[b] (clearing warp arrives, generating warps wait), b = step parity.  A generating warp
// can be at most two steps ahead of the clearing warp, so phases of one barrier never overlap.
// Same orders, same integer sums, same bytes as ks_persistent_kernel (tests).
//
// COLS = 1: one int32 per bin.  COLS = 32: the lane-columned layout -- 32 columns per bin, column =
// lane = bank, so a warp's 32 atomics never conflict; the merge adds the columns with one REDUX per
// bin.  (The aggregation ablation of SURVEY.md S7 / north_star (3); DESIGN.md 7.3 has the numbers.)
#pragma once
#include "ks_kernel.cuh"
#include <type_traits>

namespace ks {

enum { kBarFull0 = 1, kBarFree0 = 3 };     // full[b] = 1 + b, free[b] = 3 + b; barrier 0 = __syncthreads()

// barrier base + b with an immediate id in either branch (b is CTA-uniform)
template <int BASE> __device__ __forceinline__ void bar_sync_b(int b, int n) { if (b) bar_sync<BASE + 1>(n); else bar_sync<BASE>(n); }
template <int BASE> __device__ __forceinline__ void bar_arrive_b(int b, int n) { if (b) bar_arrive<BASE + 1>(n); else bar_arrive<BASE>(n); }

__device__ __forceinline__ int lds32(uint32_t saddr) { int v; asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory"); return v; }
__device__ __forceinline__ void sts32(uint32_t saddr, int v) { asm volatile("st.shared.s32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory"); }
__device__ __forceinline__ void red32(uint32_t saddr, int v) { asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory"); }

// grid = M CTAs (one per market), block = T >= 64 threads, dynamic shared memory =
// 8*L + 2 * P.rel_stride bytes: the book, then the two relative histograms.  One histogram =
// sell bins then buy bins (P.rel_side bytes each), bin i of either side <-> tick (last - delta) + i
// (ks_device.cuh, rel_bin_addr).
//
// Roles.  The CLEARING warp's loop is the serial chain of the whole run (a single warp issues a
// dependent instruction every ~5 cycles, so its length in instructions is the step time): it
// holds only what the next step needs -- take the histogram, scan, price, residual, bounds -- and
// posts (Vmax, p*, price before) in a two-slot mailbox.  The record (a6) and the trace are kept by
// the FIRST GENERATING warp, which picks the mail of step s-2 up when it passes the free[] barrier
// it waits at anyway; the last two mails are taken after the loop.
template <bool PACKED, int COLS>
__global__ void __launch_bounds__(1024, 1) ks_decoupled_kernel(const __grid_constant__ KernelParams P) {
  extern __shared__ __align__(16) int32_t book[];     // [2][L]: bid then ask; then rel[2][P.rel_stride / 4]
  __shared__ long long s_rec[16];
  __shared__ long long s_red64[64];
  __shared__ int s_red32[64];
  __shared__ int2 s_trace[32];
  __shared__ __align__(16) int s_mail[2][4];          // per step parity: Vmax, p*, price before the step
  __shared__ int s_abort;
  __shared__ int s_ovf;
  __shared__ long long s_keep[3];
  constexpr int ATOM = COLS == 1 ? 4 : 5;

  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = T >> 5;
  const int L = P.L;
  const int cw = (int)(blockIdx.x % (unsigned)nwarps);     // the clearing warp (spread over the SM's schedulers)
  const bool clearing = warp == cw;
  const uint32_t market = P.market_base + blockIdx.x;
  int32_t* gbook = P.books + (size_t)blockIdx.x * 2 * (size_t)L;
  long long* grec = P.recs + (size_t)blockIdx.x * 16;
  if (depth_check_aborts(P, &s_abort)) return;
  int32_t* rel = book + 2 * L;
  const uint32_t book_saddr = (uint32_t)__cvta_generic_to_shared(book);
  const uint32_t rel_saddr = book_saddr + 8u * (uint32_t)L;
  const int n = P.noise_n, delta = P.noise_delta;

  // ---- a0
  long long sb0, sa0;
  int bmax, amin;
  load_book(P, book, gbook, L, sb0, sa0, bmax, amin);
  for (int i = tid; i < (int)(P.rel_stride / 2); i += T) rel[i] = 0;      // both buffers
  if (tid < 16) s_rec[tid] = grec[tid];
  if (tid == 0) s_ovf = 0;
  BookTotals tot0 = block_reduce_totals(sb0, sa0, bmax, amin, s_red64, s_red32);   // has barriers
  bmax = tot0.bmax;
  amin = min(tot0.amin, L);
  int last = (int)s_rec[F_LAST];
  const uint32_t t0 = (uint32_t)s_rec[F_STEPS];
  const uint32_t S = (uint32_t)P.S;
  if (tid == 0) { s_keep[0] = tot0.sum_bid; s_keep[1] = tot0.sum_ask; s_keep[2] = s_rec[F_SUMVOL]; }
  __syncthreads();
  const int gtid = tid - (warp > cw ? 32 : 0);             // generating threads: 0 .. T-33, the clearing warp left out
  const bool bookkeeper = !clearing && gtid < 32;          // the first generating warp keeps the record and the trace
  auto take_mail = [&](uint32_t s_of_mail) {               // a6 (+ trace) of one cleared step, in step order
    const int4 m = *reinterpret_cast<const int4*>(s_mail[s_of_mail & 1u]);
    update_record_lanes(s_rec, &s_ovf, lane, m.z, m.x, m.y, m.z);
    if (P.trace) trace_step(s_trace, P.trace + (size_t)blockIdx.x * (size_t)S, (long long)s_of_mail, (long long)S, lane,
                            m.x > 0 ? m.y : m.z, m.x);
    __syncwarp();
  };

  if (clearing) {
    const LocalBook io{book, L};
    const unsigned FULL = 0xffffffffu;
    // lane masks of the 5-step scans (all-ones where the shuffled value is in range)
    int mdn[5], mup[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) { mdn[k] = lane + (1 << k) < 32 ? -1 : 0; mup[k] = lane >= (1 << k) ? -1 : 0; }
    for (uint32_t s = 0; s < S; ++s) {
      const int buf = (int)(s & 1u);
      const uint32_t rs = rel_saddr + (uint32_t)buf * P.rel_stride;   // sell bins of this step's histogram
      const uint32_t rb = rs + P.rel_side;                           // buy bins
      const int t_lo = last - delta;                       // tick of bin 0
      const int lo = max(0, min(amin, t_lo));
      const int hi = min(L - 1, max(bmax, last + delta));
      const bool inside = t_lo >= 0 && last + delta <= L - 1;   // no order of this step is clamped
      int vmax, pstar, nb, na;
      bar_sync_b<kBarFull0>(buf, T);                       // every order of step s is in the histogram
      if (COLS == 1 && inside && !P.force_generic && hi - lo < 32) {
        // ---- a2 (second half) fused into a3-a5, one tick per lane, raw shared addresses:
        // a lane adds its tick's two bins to the depth it scans (clear_window1's definitions)
        const int tick = lo + lane, i = tick - t_lo;       // this lane's tick and bin
        const bool in = tick < L, has = (unsigned)i < (unsigned)n;
        const uint32_t pb = book_saddr + 4u * (uint32_t)tick, pa = pb + 4u * (uint32_t)L;
        const int b0 = in ? lds32(pb) : 0, a0 = in ? lds32(pa) : 0;
        const int inc_a = has ? lds32(rs + 4u * (uint32_t)i) : 0, inc_b = has ? lds32(rb + 4u * (uint32_t)i) : 0;
        if (inc_a != 0) sts32(rs + 4u * (uint32_t)i, 0);
        if (inc_b != 0) sts32(rb + 4u * (uint32_t)i, 0);
        int b = b0 + inc_b, a = a0 + inc_a;
        int D = b, Sc = a;                                 // inclusive suffix of bids / prefix of asks over lanes
#pragma unroll
        for (int k = 0; k < 5; ++k) {
          const int vb = __shfl_down_sync(FULL, D, 1 << k), va = __shfl_up_sync(FULL, Sc, 1 << k);
          D += vb & mdn[k];
          Sc += va & mup[k];
        }
        const int V = min(D, Sc);
        vmax = __reduce_max_sync(FULL, V);
        pstar = __reduce_min_sync(FULL, (V == vmax && vmax > 0) ? tick : 0x7fffffff);
        if (vmax > 0) { b = min(b, max(0, D - vmax)); a = min(a, max(0, Sc - vmax)); }
        if (in && b != b0) sts32(pb, b);
        if (in && a != a0) sts32(pa, a);
        if (lane == 0) *reinterpret_cast<int4*>(s_mail[buf]) = make_int4(vmax, pstar, last, 0);
        __syncwarp();
        if (s + 2 < S) bar_arrive_b<kBarFree0>(buf, T);    // histogram empty again, mail posted: step s+2 may start
        nb = __reduce_max_sync(FULL, b > 0 ? tick : -1);
        na = __reduce_min_sync(FULL, a > 0 ? tick : 0x7fffffff);
        if (nb < 0) nb = lo - 1;
        if (na == 0x7fffffff) na = min(L, lo + 32);
      } else {
        int base, wend;
        LaneBounds lbnd;
        if (COLS == 1 && inside && !P.force_generic && hi - (lo & ~3) + 1 <= 128) {
          base = lo & ~3; wend = min(L, base + 128);
          int ib[4], ia[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int i = base + 4 * lane + j - t_lo;
            const bool has = (unsigned)i < (unsigned)n;
            ia[j] = has ? lds32(rs + 4u * (uint32_t)i) : 0; ib[j] = has ? lds32(rb + 4u * (uint32_t)i) : 0;
            if (ia[j] != 0) sts32(rs + 4u * (uint32_t)i, 0);
            if (ib[j] != 0) sts32(rb + 4u * (uint32_t)i, 0);
          }
          clear_window<4, LocalBook, true>(io, L, base, lane, vmax, pstar, lbnd, ib, ia);
        } else {
          // ---- general merge: bins -> clamped ticks, into the combined book; then the usual clearing
          if (COLS == 1) {
            for (int i = lane; i < n; i += 32) {
              const int va = lds32(rs + 4u * (uint32_t)i), vb = lds32(rb + 4u * (uint32_t)i);
              const int tick = clamp_tick(t_lo + i, L);
              if (va != 0) { sts32(rs + 4u * (uint32_t)i, 0); red32(book_saddr + 4u * (uint32_t)(tick + L), va); }
              if (vb != 0) { sts32(rb + 4u * (uint32_t)i, 0); red32(book_saddr + 4u * (uint32_t)tick, vb); }
            }
          } else {
            // lane-columned bins: 8 bins at a time (independent loads), one REDUX per bin and side
            for (int i0 = 0; i0 < n; i0 += 8) {
              int va[8], vb[8];
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                const bool has = i0 + j < n;
                va[j] = has ? lds32(rs + 128u * (uint32_t)(i0 + j) + 4u * (uint32_t)lane) : 0;
                vb[j] = has ? lds32(rb + 128u * (uint32_t)(i0 + j) + 4u * (uint32_t)lane) : 0;
              }
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                if (i0 + j < n) {
                  if (va[j] != 0) sts32(rs + 128u * (uint32_t)(i0 + j) + 4u * (uint32_t)lane, 0);
                  if (vb[j] != 0) sts32(rb + 128u * (uint32_t)(i0 + j) + 4u * (uint32_t)lane, 0);
                  const int ta = __reduce_add_sync(FULL, va[j]), tb = __reduce_add_sync(FULL, vb[j]);
                  const int tick = clamp_tick(t_lo + i0 + j, L);
                  if (lane == 0 && ta != 0) red32(book_saddr + 4u * (uint32_t)(tick + L), ta);
                  if (lane == 1 && tb != 0) red32(book_saddr + 4u * (uint32_t)tick, tb);
                }
              }
            }
          }
          __syncwarp();
          clear_active_window(io, L, lo, hi, P.force_generic != 0, lane, vmax, pstar, lbnd, base, wend);
        }
        if (lane == 0) *reinterpret_cast<int4*>(s_mail[buf]) = make_int4(vmax, pstar, last, 0);
        __syncwarp();
        if (s + 2 < S) bar_arrive_b<kBarFree0>(buf, T);
        reduce_bounds(lbnd, base, wend, nb, na);
      }
      bmax = nb; amin = na;
      last = vmax > 0 ? pstar : last;
    }
  } else {
    // ---- a1 + a2 (first half) by the generating threads
    const MarketUniform mu = market_uniform(P, market);
    const GenPlan<0> gplan = gen_plan<0>(PACKED ? (uint32_t)P.A >> 2 : (uint32_t)P.A, gtid, T - 32);
    // the most agents any generating thread holds (CTA-uniform); <= 4 takes the latency path
    const uint32_t nmax = PACKED ? 99u : gplan.cls[0].n_uniform + ((uint32_t)P.A % (uint32_t)(T - 32) != 0u ? 1u : 0u);
    BookRef bref; bref.ptr = book; bref.saddr = 0;
    RuleCtx rc;
    rc.last = 0; rc.dp = 0; rc.L = L; rc.noclamp = true; rc.bid_lo = 0; rc.ask_lo = 0; rc.bid_last = 0; rc.ask_last = 0;
    rc.mid2 = 0; rc.mkt_flags = nullptr;
    const uint32_t col = COLS == 32 ? 4u * (uint32_t)lane : 0u;
    const uint32_t bin_bytes = COLS == 32 ? 128u : 4u;
    int sink = 0;
    for (uint32_t s = 0; s < S; ++s) {
      const int buf = (int)(s & 1u);
      const StepUniform u = step_uniform(P, mu, t0 + s);
      rc.rel_s = rel_saddr + (uint32_t)buf * P.rel_stride + col;
      rc.rel_b = rc.rel_s + P.rel_side + (uint32_t)(n - 1) * bin_bytes;
      if (s >= 2) {
        bar_sync_b<kBarFree0>(buf, T);                     // the clearing warp has drained this histogram (step s-2)
        if (bookkeeper) take_mail(s - 2);
      }
      if (nmax == 1u)      generate_class_rel_few<ATOM, 1>(P, bref, mu, u, rc, gplan.cls[0], gplan.p0_inc, sink);
      else if (nmax == 2u) generate_class_rel_few<ATOM, 2>(P, bref, mu, u, rc, gplan.cls[0], gplan.p0_inc, sink);
      else if (nmax == 3u) generate_class_rel_few<ATOM, 3>(P, bref, mu, u, rc, gplan.cls[0], gplan.p0_inc, sink);
      else if (nmax == 4u) generate_class_rel_few<ATOM, 4>(P, bref, mu, u, rc, gplan.cls[0], gplan.p0_inc, sink);
      else                 generate_step<0, ATOM, PACKED>(P, bref, mu, u, rc, gplan, gtid == 0, sink);
      bar_arrive_b<kBarFull0>(buf, T);
    }
  }
  __syncthreads();                                         // the last clearing is done
  if (bookkeeper) {                                        // the mails of the last two steps
    if (S >= 2) take_mail(S - 2);
    if (S >= 1) take_mail(S - 1);
  }

  // ---- a7 (its first block barrier publishes the bookkeeper's record)
  store_state(P, book, gbook, grec, L, s_rec, s_keep, &s_ovf, s_red64, s_red32);
}

}  // namespace ks
