// ks_decoupled.cuh -- order generation DECOUPLED from the clearing price.
//
// In ks_persistent_kernel a step is a chain: generate (needs the price) | barrier | clear (gives
// the next price) | barrier.  When many markets share an SM and every market brings many agents
// (C4), the markets hide each other's chains; with few markets per SM (C2: 7) or one (C3, C1) the
// chain IS the run time: while one warp clears, the market's other warps idle at the barrier
// (ncu on C2, profiles/r2a_c2_persistent.md: 42 % of all warp samples).  But for a
// zero-intelligence agent only the TICK depends on the price, not the order: offset draw o, side
// and quantity are pure functions of (seed, market, step, agent).  So here the generating warps
// never see a price.  They add their orders to a relative histogram (sell[o], buy[n-1-o]: bin i of
// either side means tick last - delta + i; ATOM 4 / 5 of ks_device.cuh) taken from a RING of NB
// histograms, and run up to NB steps ahead; ONE clearing warp per market (which holds no agents)
// takes histogram s mod NB at the current price -- exactly the rule's ticks, clamped to the grid --
// zeroes it, hands it back, and clears (a3-a6).  In the common case (no order clamped, window <=
// 128 ticks) the histogram is not even merged into the book first: each lane adds its ticks' bins
// to the depth it loads for the scan.  With a ring deep enough to absorb the hand-over latency
// (measured: a two-deep ring leaves BOTH sides waiting for each other a third of the time) the
// step time is max(generate, clear), and the SM's warps never idle at a barrier.
//
// Synchronisation: 2*NB named barriers, full[b] (generating warps arrive, clearing warp waits)
// and free[b] (clearing warp arrives, generating warps wait), b = step mod NB.  A generating warp
// can be at most NB steps ahead of the clearing warp, so phases of one barrier never overlap.
// Same orders, same integer sums, same bytes as ks_persistent_kernel (tests).
//
// COLS = 1: one int32 per bin.  COLS = 32: the lane-columned layout -- 32 columns per bin, column =
// lane = bank, so a warp's 32 atomics never conflict; the merge adds the columns with one REDUX per
// bin.  (The aggregation ablation of SURVEY.md S7 / north_star (3); DESIGN.md 7.3 has the numbers.)
#pragma once
#include "ks_kernel.cuh"
#include <type_traits>

namespace ks {

// barrier ids: full[b] = 1 + b, free[b] = 1 + NB + b; barrier 0 = __syncthreads().  The id must be
// an immediate (ks_kernel.cuh), hence the switch over the CTA-uniform b.
template <int BASE, int NB> __device__ __forceinline__ void bar_sync_b(int b, int n) {
  static_assert(NB == 2 || NB == 4, "ring depth");
  if (NB == 2) { if (b) bar_sync<BASE + 1>(n); else bar_sync<BASE>(n); }
  else {
    switch (b) {
      case 0: bar_sync<BASE>(n); break;
      case 1: bar_sync<BASE + 1>(n); break;
      case 2: bar_sync<BASE + (NB > 2 ? 2 : 0)>(n); break;
      default: bar_sync<BASE + (NB > 2 ? 3 : 1)>(n); break;
    }
  }
}
template <int BASE, int NB> __device__ __forceinline__ void bar_arrive_b(int b, int n) {
  if (NB == 2) { if (b) bar_arrive<BASE + 1>(n); else bar_arrive<BASE>(n); }
  else {
    switch (b) {
      case 0: bar_arrive<BASE>(n); break;
      case 1: bar_arrive<BASE + 1>(n); break;
      case 2: bar_arrive<BASE + (NB > 2 ? 2 : 0)>(n); break;
      default: bar_arrive<BASE + (NB > 2 ? 3 : 1)>(n); break;
    }
  }
}

__device__ __forceinline__ int lds32(uint32_t saddr) { int v; asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory"); return v; }
__device__ __forceinline__ void sts32(uint32_t saddr, int v) { asm volatile("st.shared.s32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory"); }
__device__ __forceinline__ void red32(uint32_t saddr, int v) { asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(saddr), "r"(v) : "memory"); }

// grid = M CTAs (one per market), block = T >= 64 threads (<= MAXT), dynamic shared memory =
// 8*L + NB * P.rel_stride bytes: the book, then the ring of NB relative histograms.  One histogram
// = sell bins then buy bins (P.rel_side bytes each), bin i of either side <-> tick (last - delta) + i
// (ks_device.cuh, rel_bin_addr).  MAXT / MINB: launch bounds (the register budget that lets MINB
// CTAs of MAXT threads share an SM -- C2 needs 7 markets of 160 threads resident per SM).
//
// Roles.  The CLEARING warp's loop is the serial chain of the whole run (a single warp issues a
// dependent instruction every ~5-10 cycles, so its length in instructions is the step time): it
// holds only what the next step needs -- take the histogram, scan, price, residual, bounds -- and
// posts (Vmax, p*, price before) in an NB-slot mailbox.  The record (a6) and the trace are kept by
// the FIRST GENERATING warp, which picks the mail of step s-NB up when it passes the free[]
// barrier it waits at anyway; the last NB mails are taken after the loop.
// MIX: the three-type population (KS_MODEL_MIX3) -- every rule expressed relative to the price the
// step starts from (generate_mix3_rel_group); the clearing warp merges the bins at the step's price
// and price change.  Only with GROUP steps per hand-over.
template <bool PACKED, int COLS, int NB, int MAXT, int MINB, int GROUP = 1, bool MIX = false>
__global__ void __launch_bounds__(MAXT, MINB) ks_decoupled_kernel(const __grid_constant__ KernelParams P) {
  constexpr bool PAIR = GROUP > 1;      // GROUP = 2 or 4 steps per pass over the agents and per hand-over
  static_assert(!PAIR || (NB == 2 * GROUP && COLS == 1 && !PACKED), "GROUP steps per hand-over: ring of 2*GROUP, literal contract");
  static_assert(!MIX || PAIR, "MIX3 runs with GROUP steps per hand-over only");
  extern __shared__ __align__(16) int32_t book[];     // [2][L]: bid then ask; then rel[NB][P.rel_stride / 4]
  __shared__ long long s_rec[16];
  __shared__ long long s_red64[64];
  __shared__ int s_red32[64];
  __shared__ int2 s_trace[32];
  __shared__ __align__(16) int s_mail[NB][4];         // per ring slot: Vmax, p*, price before the step
  __shared__ int s_abort;
  __shared__ int s_ovf;
  __shared__ long long s_keep[3];
  constexpr int ATOM = COLS == 1 ? 4 : 5;
#ifdef KS_DEBUG_CHECKS
  __shared__ int s_dbg_count[NB];                     // orders added to each ring slot since it was last drained
  if (threadIdx.x < NB) s_dbg_count[threadIdx.x] = 0;
#endif
  constexpr int kBarFull0 = 1, kBarFree0 = 1 + NB;

  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = T >> 5;
  const int L = P.L;
  // The clearing warp is the LAST warp and the block has 4k+1 warps (ks_api.cu): warps map to the
  // SM's four schedulers by index, so the 4k generating warps load the schedulers evenly and the
  // clearing warp shares scheduler 0 (measured on C2: with the clearing warp rotating over the
  // warp indices, scheduler 0 carried two generating warps of most markets: 4.1 ms vs 3.6 ms).
  const int cw = nwarps - 1;
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
  for (int i = tid; i < (int)(NB * (P.rel_stride / 4)); i += T) rel[i] = 0;      // the whole ring
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
  // Who keeps the record (a6) and the trace.  Latency regime (C1, C3): the clearing warp's chain IS
  // the step time, so the first generating warp does it from the mailbox.  Throughput regime (the
  // (160, 7) two-deep-ring instantiation, C2): the SM is bound by dispatched instructions and the
  // clearing warp has slack (it waits at full[] 40 % of its time), so it does the bookkeeping itself,
  // straight from its registers: no mailbox round trip, and the four generating warps stay equal.
  constexpr bool kClearingKeepsBooks = (MAXT <= 160 && NB == 2) || PAIR;
  const bool bookkeeper = kClearingKeepsBooks ? clearing : warp == 0;
  long long rec_reg = s_rec[lane & 15];                    // ... lane f (and f + 16) holding field f in a register
  int ovf_reg = 0;
  auto take_mail = [&](uint32_t s_of_mail, int slot) {     // a6 (+ trace) of one cleared step, in step order
    const int4 m = *reinterpret_cast<const int4*>(s_mail[slot]);
    update_record_reg(rec_reg, ovf_reg, lane, m.z, m.x, m.y, m.z);
    if (P.trace) trace_step(s_trace, P.trace + (size_t)blockIdx.x * (size_t)S, (long long)s_of_mail, (long long)S, lane,
                            m.x > 0 ? m.y : m.z, m.x);
  };

  if (clearing) {
    const LocalBook io{book, L};
    const unsigned FULL = 0xffffffffu;
    int prevp = (int)s_rec[F_PREV];                      // MIX3: the price before `last` (momentum's side)
#ifdef KS_DEBUG_CHECKS
    int dbg_steps = 1;                                   // steps handed over with the group being cleared
#endif
    // a2 (second half) + a3-a5 of one step on the histogram whose sell bins start at rs (ring slot
    // `slot`); wait() is called where the histogram is first needed
    auto clear_core = [&](uint32_t rs, int slot, auto wait, int& vmax, int& pstar, int& base, int& wend, LaneBounds& lbnd) {
      (void)slot;
      const uint32_t rb = rs + P.rel_side;                           // buy bins
      const int t_lo = last - delta;                     // tick of bin 0
      const int lo = max(0, min(amin, t_lo));
      const int hi = min(L - 1, max(bmax, last + delta));
      const bool inside = t_lo >= 0 && last + delta <= L - 1;   // no order of this step is clamped
      [[maybe_unused]] const bool fuse = COLS == 1 && inside && !P.force_generic;
      wait();                                            // every order of this step is in the histogram
#ifdef KS_DEBUG_CHECKS
      // (GROUP steps per hand-over: the whole group's orders are counted in its first slot's counter and
      // checked when its first step is cleared)
      if (lane == 0 && !MIX && (!PAIR || slot % GROUP == 0)) {
        const int steps_here = PAIR ? dbg_steps : 1;
        KS_CHECK(s_dbg_count[slot] == steps_here * P.A, "orders in the histogram(s) at full[] != agents x steps handed over");
        s_dbg_count[slot] = 0;
      }
      __syncwarp();
#endif
      if constexpr (MIX) {
        // ---- MIX3 merge: every bin -> its clamped tick(s) in the combined book, then the usual clearing.
        // noise: bin i of either side <-> tick last - delta + i
        for (int i = lane; i < n; i += 32) {
          const int va = lds32(rs + 4u * (uint32_t)i), vb = lds32(rb + 4u * (uint32_t)i);
          const int tick = clamp_tick(t_lo + i, L);
          if (va != 0) { sts32(rs + 4u * (uint32_t)i, 0); red32(book_saddr + 4u * (uint32_t)(tick + L), va); }
          if (vb != 0) { sts32(rb + 4u * (uint32_t)i, 0); red32(book_saddr + 4u * (uint32_t)tick, vb); }
        }
        // makers: bin s0 -> bid at last - 1 - s0 AND ask at last + 1 + s0
        for (int i = lane; i < P.maker_spread_max; i += 32) {
          const uint32_t a = rs + P.rel_mk_off + 4u * (uint32_t)i;
          const int v = lds32(a);
          if (v != 0) {
            sts32(a, 0);
            red32(book_saddr + 4u * (uint32_t)clamp_tick(last - 1 - i, L), v);
            red32(book_saddr + 4u * (uint32_t)(clamp_tick(last + 1 + i, L) + L), v);
          }
        }
        // momentum: side = sgn(last - prev) of the step being cleared; the coin bins decide a flat price
        const int dp = last - prevp;
        for (int i = lane; i < P.mom_n; i += 32) {
          const uint32_t a = rs + P.rel_mom_off + 4u * (uint32_t)i;
          const int vall = lds32(a), vcoin = lds32(a + P.rel_mom_side);
          if (vall != 0) sts32(a, 0);
          if (vcoin != 0) sts32(a + P.rel_mom_side, 0);
          const int vbuy = dp > 0 ? vall : (dp < 0 ? 0 : vcoin), vsell = vall - vbuy;
          if (vbuy != 0) red32(book_saddr + 4u * (uint32_t)clamp_tick(last + i, L), vbuy);
          if (vsell != 0) red32(book_saddr + 4u * (uint32_t)(clamp_tick(last - i, L) + L), vsell);
        }
        __syncwarp();
        clear_active_window(io, L, max(0, min(amin, last - P.dmax)), min(L - 1, max(bmax, last + P.dmax)), P.force_generic != 0,
                            lane, vmax, pstar, lbnd, base, wend);
      } else if (fuse && hi - lo < 32) {
        // this lane's bins of tick lo + lane (a2, second half): read and zeroed here, added to the
        // depth inside the scan
        int ib[1], ia[1];
        base = lo; wend = min(L, lo + 32);
        const int i = lo + lane - t_lo;
        const bool has = (unsigned)i < (unsigned)n;
        ia[0] = has ? lds32(rs + 4u * (uint32_t)i) : 0; ib[0] = has ? lds32(rb + 4u * (uint32_t)i) : 0;
        if (ia[0] != 0) sts32(rs + 4u * (uint32_t)i, 0);
        if (ib[0] != 0) sts32(rb + 4u * (uint32_t)i, 0);
        clear_rows<1, LocalBook, true>(io, L, base, lane, vmax, pstar, lbnd, ib, ia);
      } else if (fuse && hi - lo < 64) {
        int ib[2], ia[2];
        base = lo; wend = min(L, lo + 64);
#pragma unroll
        for (int r = 0; r < 2; ++r) {
          const int i = lo + 32 * r + lane - t_lo;
          const bool has = (unsigned)i < (unsigned)n;
          ia[r] = has ? lds32(rs + 4u * (uint32_t)i) : 0; ib[r] = has ? lds32(rb + 4u * (uint32_t)i) : 0;
          if (ia[r] != 0) sts32(rs + 4u * (uint32_t)i, 0);
          if (ib[r] != 0) sts32(rb + 4u * (uint32_t)i, 0);
        }
        clear_rows<2, LocalBook, true>(io, L, base, lane, vmax, pstar, lbnd, ib, ia);
      } else if (fuse && hi - (lo & ~3) + 1 <= 128) {
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
    };
    if constexpr (!PAIR) {
    for (uint32_t s0 = 0; s0 < S; s0 += NB) {
#pragma unroll
        for (int buf = 0; buf < NB; ++buf) {                 // ring slot = step mod NB, a compile-time constant here
          const uint32_t s = s0 + (uint32_t)buf;
          if (s >= S) break;
          int vmax, pstar, base, wend;
          LaneBounds lbnd;
          clear_core(rel_saddr + (uint32_t)buf * P.rel_stride, buf, [&] { bar_sync_b<kBarFull0, NB>(buf, T); }, vmax, pstar, base, wend, lbnd);
          if (!kClearingKeepsBooks) {
            if (lane == 0) *reinterpret_cast<int4*>(s_mail[buf]) = make_int4(vmax, pstar, last, 0);
          }
          __syncwarp();
          if (s + NB < S) bar_arrive_b<kBarFree0, NB>(buf, T);   // histogram empty again, mail posted: step s+NB may start
          if (kClearingKeepsBooks) {
            update_record_reg(rec_reg, ovf_reg, lane, last, vmax, pstar, last);
            if (P.trace) trace_step(s_trace, P.trace + (size_t)blockIdx.x * (size_t)S, (long long)s, (long long)S, lane,
                                    vmax > 0 ? pstar : last, vmax);
          }
          int nb, na;
          reduce_bounds(lbnd, base, wend, nb, na);
          bmax = nb; amin = na;
          last = vmax > 0 ? pstar : last;
        }
      }
    }
    if constexpr (PAIR) {
      // GROUP steps per hand-over: ring slots GROUP*p .. GROUP*p + GROUP-1 belong to group p = (s / GROUP) mod 2;
      // one full[p] / free[p] barrier per group (ids: full 1 + p, free 3 + p); the steps of a group are
      // cleared by a rolled loop
      for (uint32_t s0 = 0; s0 < S; s0 += 2 * GROUP) {
#pragma unroll
        for (int pr = 0; pr < 2; ++pr) {
          const uint32_t s = s0 + (uint32_t)(GROUP * pr);
          if (s >= S) break;
          const uint32_t ns = min((uint32_t)GROUP, S - s);
#ifdef KS_DEBUG_CHECKS
          dbg_steps = (int)ns;
#endif
          for (uint32_t g = 0; g < ns; ++g) {
            const int slot = GROUP * pr + (int)g;
            int vmax, pstar, base, wend;
            LaneBounds lbnd;
            clear_core(rel_saddr + (uint32_t)slot * P.rel_stride, slot, [&] { if (g == 0) bar_sync_b<1, 2>(pr, T); }, vmax, pstar, base, wend, lbnd);
            if (g + 1 == ns) {
              __syncwarp();
              if (s + 2 * GROUP < S) bar_arrive_b<3, 2>(pr, T);   // the group's histograms are empty again
            }
            update_record_reg(rec_reg, ovf_reg, lane, last, vmax, pstar, last);
            if (P.trace) trace_step(s_trace, P.trace + (size_t)blockIdx.x * (size_t)S, (long long)(s + g), (long long)S, lane,
                                    vmax > 0 ? pstar : last, vmax);
            int nb, na;
            reduce_bounds(lbnd, base, wend, nb, na);
            bmax = nb; amin = na;
            prevp = last;
            last = vmax > 0 ? pstar : last;
          }
        }
      }
    }
  } else {
    // ---- a1 + a2 (first half) by the generating threads tid 0 .. T-33
    const MarketUniform mu = market_uniform(P, market);
    const GenPlan<0> gplan = gen_plan<0>(PACKED ? (uint32_t)P.A >> 2 : (uint32_t)P.A, tid, T - 32);
    const GenPlan<1> gplan3 = gen_plan<1>((uint32_t)P.A, tid, T - 32);     // MIX3: agent 3j + c has type c
    // the most agents any generating thread holds (CTA-uniform); <= 4 takes the latency path
    const uint32_t nmax = PACKED ? 99u : gplan.cls[0].n_uniform + ((uint32_t)P.A % (uint32_t)(T - 32) != 0u ? 1u : 0u);
    BookRef bref; bref.ptr = book; bref.saddr = 0;
    RuleCtx rc;
    rc.last = 0; rc.dp = 0; rc.L = L; rc.noclamp = true; rc.bid_lo = 0; rc.ask_lo = 0; rc.bid_last = 0; rc.ask_last = 0;
    rc.mid2 = 0; rc.mkt_flags = nullptr;
    const uint32_t col = COLS == 32 ? 4u * (uint32_t)lane : 0u;
    const uint32_t bin_bytes = COLS == 32 ? 128u : 4u;
    int sink = 0;
    if constexpr (PAIR) {
      // GROUP steps per pass over the agents: for one agent the Philox rounds that do not depend on
      // the step (M0*a, M1*n2, M0*c0: two multiplies and two xors of rounds 0-2) and the counter add
      // are shared by the GROUP steps, and the per-step prologue of the loop is paid once per group
      for (uint32_t s0 = 0; s0 < S; s0 += 2 * GROUP) {
#pragma unroll
        for (int pr = 0; pr < 2; ++pr) {
          const uint32_t s = s0 + (uint32_t)(GROUP * pr);
          if (s >= S) break;
          const uint32_t slot0 = rel_saddr + (uint32_t)(GROUP * pr) * P.rel_stride;
          if (s0 != 0u) bar_sync_b<3, 2>(pr, T);           // free[pr]: the clearing warp has drained the group's histograms
          if (s + GROUP <= S) {
            StepUniform ug[GROUP];
#pragma unroll
            for (int g = 0; g < GROUP; ++g) ug[g] = step_uniform(P, mu, t0 + s + (uint32_t)g);
#ifdef KS_DEBUG_CHECKS
            bref.dbg_lo = slot0; bref.dbg_hi = slot0 + GROUP * P.rel_stride; bref.dbg_count = &s_dbg_count[GROUP * pr];
#endif
            if constexpr (MIX)
              generate_mix3_rel_group<GROUP>(P, bref, mu, ug, slot0, P.rel_stride, P.rel_side + (uint32_t)(n - 1) * 4u, gplan3, sink);
            else
              generate_class_rel_group<ATOM, GROUP>(P, bref, mu, ug, slot0, P.rel_stride, P.rel_side + (uint32_t)(n - 1) * 4u,
                                                    gplan.cls[0], gplan.p0_inc, sink);
          } else {                                         // the run's last, partial group: step by step
            for (uint32_t g = 0; s + g < S; ++g) {
              const StepUniform u = step_uniform(P, mu, t0 + s + g);
              rc.rel_s = slot0 + g * P.rel_stride;
              rc.rel_b = rc.rel_s + P.rel_side + (uint32_t)(n - 1) * 4u;
#ifdef KS_DEBUG_CHECKS
              bref.dbg_lo = rc.rel_s; bref.dbg_hi = bref.dbg_lo + P.rel_stride; bref.dbg_count = &s_dbg_count[GROUP * pr];
#endif
              if constexpr (MIX) {
                const StepUniform u1[1] = {u};
                generate_mix3_rel_group<1>(P, bref, mu, u1, rc.rel_s, P.rel_stride, P.rel_side + (uint32_t)(n - 1) * 4u, gplan3, sink);
              } else {
                generate_step<0, ATOM, PACKED>(P, bref, mu, u, rc, gplan, tid == 0, sink);
              }
            }
          }
          bar_arrive_b<1, 2>(pr, T);                       // full[pr]
        }
      }
    }
    // the whole step loop, instantiated per N = events a thread holds (0 = the general loop), so that
    // nothing about N is decided inside it
    auto gen_loop = [&](auto Ntag) {
      constexpr int N = decltype(Ntag)::value;
      for (uint32_t s0 = 0; s0 < S; s0 += NB) {
#pragma unroll
        for (int buf = 0; buf < NB; ++buf) {
          const uint32_t s = s0 + (uint32_t)buf;
          if (s >= S) break;
          const StepUniform u = step_uniform(P, mu, t0 + s);
          rc.rel_s = rel_saddr + (uint32_t)buf * P.rel_stride + col;
          rc.rel_b = rc.rel_s + P.rel_side + (uint32_t)(n - 1) * bin_bytes;
#ifdef KS_DEBUG_CHECKS
          bref.dbg_lo = rel_saddr + (uint32_t)buf * P.rel_stride; bref.dbg_hi = bref.dbg_lo + P.rel_stride;
          bref.dbg_count = &s_dbg_count[buf];
#endif
          if (s0 != 0u) {
            bar_sync_b<kBarFree0, NB>(buf, T);             // the clearing warp has drained this histogram (step s-NB)
            if (!kClearingKeepsBooks && bookkeeper) take_mail(s - (uint32_t)NB, buf);
          }
          if constexpr (N > 0) generate_class_rel_few<ATOM, N>(P, bref, mu, u, rc, gplan.cls[0], gplan.p0_inc, sink);
          else                 generate_step<0, ATOM, PACKED>(P, bref, mu, u, rc, gplan, tid == 0, sink);
          bar_arrive_b<kBarFull0, NB>(buf, T);
        }
      }
    };
    if constexpr (!PAIR) {
      if (nmax == 1u)      gen_loop(std::integral_constant<int, 1>{});
      else if (nmax == 2u) gen_loop(std::integral_constant<int, 2>{});
      else if (nmax == 3u) gen_loop(std::integral_constant<int, 3>{});
      else if (nmax == 4u) gen_loop(std::integral_constant<int, 4>{});
      else                 gen_loop(std::integral_constant<int, 0>{});
    }
  }
  __syncthreads();                                         // the last clearing is done
  if (bookkeeper) {                                        // the mails of the last NB steps, then the record goes back
    if (!kClearingKeepsBooks)
      for (uint32_t s = S > (uint32_t)NB ? S - (uint32_t)NB : 0u; s < S; ++s) take_mail(s, (int)(s & (uint32_t)(NB - 1)));
    if (lane < 16) s_rec[lane] = rec_reg;
    if (ovf_reg) s_ovf = 1;
  }

  // ---- a7 (its first block barrier publishes the bookkeeper's record)
  store_state(P, book, gbook, grec, L, s_rec, s_keep, &s_ovf, s_red64, s_red32);
}

}  // namespace ks
