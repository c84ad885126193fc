// ks_kernel.cuh -- the persistent kernel (a0-a7) and the state-initialisation kernel.
#pragma once
#include "ks_device.cuh"

namespace ks {

// Block-wide reduction of (sum, sum, max, min) used once at load and once at write-back.
struct BookTotals { long long sum_bid, sum_ask; int bmax, amin; };

__device__ __forceinline__ BookTotals block_reduce_totals(long long sb, long long sa, int bmax, int amin,
                                                          long long* s_red64, int* s_red32) {
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    sb += __shfl_xor_sync(FULL, sb, d);
    sa += __shfl_xor_sync(FULL, sa, d);
  }
  bmax = __reduce_max_sync(FULL, bmax);
  amin = __reduce_min_sync(FULL, amin);
  __syncthreads();                      // protect s_red* against a previous use
  if (lane == 0) { s_red64[2 * warp] = sb; s_red64[2 * warp + 1] = sa; s_red32[2 * warp] = bmax; s_red32[2 * warp + 1] = amin; }
  __syncthreads();
  BookTotals r; r.sum_bid = 0; r.sum_ask = 0; r.bmax = -1; r.amin = 0x7fffffff;
  for (int w = 0; w < nwarps; ++w) {
    r.sum_bid += s_red64[2 * w]; r.sum_ask += s_red64[2 * w + 1];
    r.bmax = max(r.bmax, s_red32[2 * w]); r.amin = min(r.amin, s_red32[2 * w + 1]);
  }
  return r;
}

// a6: price state, statistics and trajectory hash -- executed by lane 0 of warp 0 on the
// shared-memory copy of the record (include/kineticsim.h, ks_market_stats).
__device__ __forceinline__ void update_record(long long* rec, int last, int vmax, int pstar, int& new_last) {
  long long before = last;
  unsigned long long x;
  new_last = last;
  if (vmax > 0) {
    new_last = pstar;
    rec[F_NTRADES] += 1;
    rec[F_SUMVOL] += vmax;
    rec[F_SUMPX] += pstar;
    rec[F_SUMPX2] += (long long)pstar * pstar;
    rec[F_SUMPXVOL] += (long long)pstar * vmax;
    x = ((unsigned long long)(unsigned)vmax << 16) | (unsigned long long)(unsigned)pstar;
  } else {
    x = 0xFFFFull;
  }
  long long r = (long long)new_last - before;
  long long r2 = r * r;
  rec[F_SUMRET] += r;
  rec[F_SUMRET2] += r2;
  rec[F_SUMRET3] += r2 * r;
  rec[F_SUMRET4] += r2 * r2;
  rec[F_HASH] = (long long)(((unsigned long long)rec[F_HASH] ^ x) * kHashPrime);
  rec[F_STEPS] += 1;
  rec[F_PREV] = before;
  rec[F_LAST] = new_last;
}

// The per-thread generation plan of a launch (MODEL 2 = the paper's agent model has its own).
template <int MODEL>
__device__ __forceinline__ GenPlan<MODEL> make_gen_plan(const KernelParams& P, bool packed, int tid, int T) {
  return gen_plan<MODEL>(packed ? (uint32_t)P.A >> 2 : (uint32_t)P.A, tid, T);
}
template <>
__device__ __forceinline__ GenPlan<2> make_gen_plan<2>(const KernelParams& P, bool, int tid, int T) {
  return gen_plan_paper(P, tid, T);
}

constexpr int kPipeEvents = 4;     // PIPE kernels: events per generating thread held in registers

__device__ __forceinline__ int sign_of(int x) { return (x > 0) - (x < 0); }

// ---------------------------------------------------------------------------------------------
// The persistent kernel.  grid = M CTAs (one per market), block = T threads (any multiple of 32),
// dynamic shared memory = 8*L bytes (the book).  MODEL: 0 = ZI, 1 = MIX3, 2 = the paper's agent
// model (mid-price reference, A24).  ATOM: see book_add.
// PACKED: the PACKED4 draw contract (one Philox block per four agents, A22).
// PIPE (MODEL 0, ATOM 0, literal contract, few markets): software pipeline for the latency-bound
// regime (C3).  The Philox words of a step do not depend on the price, only the address does: warp 0
// holds no agents and only clears; while it clears step s, the other warps draw (offset, side,
// quantity) of step s+1 into registers (at most 4 events per thread), and after the barrier they
// only compute addresses and issue the atomics.  Same orders, same bytes.
// ---------------------------------------------------------------------------------------------
template <int MODEL, int ATOM, bool PACKED, bool PIPE = false>
__global__ void __launch_bounds__(1024, 1) ks_persistent_kernel(const __grid_constant__ KernelParams P) {
  extern __shared__ __align__(16) int32_t book[];     // [2][L]: bid then ask
  __shared__ long long s_rec[16];
  __shared__ long long s_red64[64];
  __shared__ int s_red32[64];
  __shared__ int2 s_trace[32];                        // staged trace entries (only when P.trace)
  __shared__ __align__(16) int s_ctl[4];              // per-step broadcast: last, &bid[last-delta], &ask[last-delta], noclamp
                                                      // (MODEL 2: last, mid2, sgn(mid2 - previous mid2), 0)
  __shared__ int s_mkt[2];                            // MODEL 2: a marketable buy / sell was generated this step

  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5;
  const int L = P.L;
  const uint32_t market = P.market_base + blockIdx.x;
  int32_t* gbook = P.books + (size_t)blockIdx.x * 2 * (size_t)L;
  long long* grec = P.recs + (size_t)blockIdx.x * 16;
  const MarketUniform mu = market_uniform(P, market);

  const GenPlan<MODEL> gplan = PIPE ? gen_plan<MODEL>(warp > 0 ? (uint32_t)P.A : 0u, tid >= 32 ? tid - 32 : 0, T - 32)
                                    : make_gen_plan<MODEL>(P, PACKED, tid, T);
  BookRef bref; bref.ptr = book; bref.saddr = (uint32_t)__cvta_generic_to_shared(book);

  // ---- a0: state load (HBM -> shared), skipped for a fresh (all-zero) book
  long long sb0 = 0, sa0 = 0;
  int bmax = -1, amin = 0x7fffffff;
  {
    const int nvec = L / 2;                            // int4 vectors in the whole book
    int4* sbook4 = reinterpret_cast<int4*>(book);
    if (P.fresh) {
      for (int i = tid; i < nvec; i += T) sbook4[i] = make_int4(0, 0, 0, 0);
    } else {
      const int4* gbook4 = reinterpret_cast<const int4*>(gbook);
      const int nside = L / 4;
      for (int i = tid; i < nvec; i += T) {
        int4 v = __ldg(gbook4 + i);
        sbook4[i] = v;
        int vals[4] = {v.x, v.y, v.z, v.w};
        if (i < nside) {
#pragma unroll
          for (int j = 0; j < 4; ++j) { sb0 += vals[j]; if (vals[j] > 0) bmax = max(bmax, 4 * i + j); }
        } else {
#pragma unroll
          for (int j = 0; j < 4; ++j) { sa0 += vals[j]; if (vals[j] > 0) amin = min(amin, 4 * (i - nside) + j); }
        }
      }
    }
    if (tid < 16) s_rec[tid] = grec[tid];
  }
  BookTotals tot0 = block_reduce_totals(sb0, sa0, bmax, amin, s_red64, s_red32);   // has barriers
  bmax = tot0.bmax;                       // only warp 0 keeps these up to date below
  amin = min(tot0.amin, L);
  int last = (int)s_rec[F_LAST], prev = (int)s_rec[F_PREV];
  const uint32_t t0 = (uint32_t)s_rec[F_STEPS];
  const long long vol0 = s_rec[F_SUMVOL];

  int sink = 0;                           // only used by the ATOM == 2 microbenchmark variant
  auto publish = [&](int new_last) {      // one thread: the rule context of the next step
    RuleCtx rc = rule_ctx(P, bref, new_last, new_last);
    *reinterpret_cast<int4*>(s_ctl) = make_int4(new_last, (int)rc.bid_lo, (int)rc.ask_lo, rc.noclamp ? 1 : 0);
  };
  // MODEL 2: Eq.3 on the exact best quotes of the resting book; f[13] holds the
  // doubled mid of the previous step
  auto publish_paper = [&](int new_last, int bb, int ba, int mid2_before) {
    const int mid2 = (bb >= 0 && ba < L) ? bb + ba : 2 * new_last;
    *reinterpret_cast<int4*>(s_ctl) = make_int4(new_last, mid2, sign_of(mid2 - mid2_before), 0);
  };
  if (tid == 0) {
    if (MODEL == 2) { publish_paper(last, bmax, amin, prev); s_mkt[0] = 0; s_mkt[1] = 0; }
    else publish(last);
  }
  __syncthreads();
  // a3-a6: clearing by warp 0 on the active window (called by warp 0 only)
  auto clear_step = [&](long long s, const RuleCtx& rc) {
    int lo, hi;
    if (MODEL == 2) {
      lo = max(0, min(amin, (rc.mid2 >> 1) - P.dmax));
      hi = min(L - 1, max(bmax, ((rc.mid2 + 1) >> 1) + P.dmax));
      if (s_mkt[0]) hi = L - 1;                      // marketable buys sit at tick L-1,
      if (s_mkt[1]) lo = 0;                          // marketable sells at tick 0
      __syncwarp();
    } else {
      lo = max(0, min(amin, last - P.dmax));
      hi = min(L - 1, max(bmax, last + P.dmax));
    }
    int vmax, pstar, nb, na, base, wend;
    int width4 = hi - (lo & ~3) + 1, width8 = hi - (lo & ~7) + 1;
    const LocalBook io{book, L};
    if (P.force_generic || width8 > 256) { base = lo & ~3; wend = min(L, hi + 1); clear_generic(io, L, base, hi, lane, vmax, pstar, nb, na); }
    else if (hi - lo < 32)               { base = lo; wend = min(L, base + 32); clear_window1(io, L, base, lane, vmax, pstar, nb, na); }
    else if (width4 <= 128)              { base = lo & ~3; wend = min(L, base + 128); clear_window<4>(io, L, base, lane, vmax, pstar, nb, na); }
    else                                 { base = lo & ~7; wend = min(L, base + 256); clear_window<8>(io, L, base, lane, vmax, pstar, nb, na); }
    if (MODEL == 2) {
      // the mid price needs the EXACT best quotes: a side with no depth inside the window is
      // searched outside it (rare: the window was emptied on that side)
      if (nb < base) nb = best_bid_below(io, L, base, lane);
      if (na >= wend) na = best_ask_from(io, L, wend, lane);
    }
    bmax = nb; amin = na;
    if (lane == 0) {
      int new_last;
      update_record(s_rec, last, vmax, pstar, new_last);
      if (MODEL == 2) {
        s_rec[F_PREV] = rc.mid2;
        publish_paper(new_last, nb, na, rc.mid2);
        s_mkt[0] = 0; s_mkt[1] = 0;
      } else {
        publish(new_last);
      }
    }
    if (P.trace) trace_step(s_trace, P.trace + (size_t)blockIdx.x * (size_t)P.S, s, P.S, lane,
                            vmax > 0 ? pstar : last, vmax);
  };
  // ---- S steps, all on-chip
  if constexpr (PIPE) {
    // per-thread draws of ONE step: the offset index o = mulhi(w1, n), and q with the side bit of
    // w0 in its top bit (q <= 2^20 + 1).  At most kPipeEvents events per thread (host plan).
    uint32_t dr_o[kPipeEvents], dr_q[kPipeEvents];
    const int n_mine = (int)gplan.cls[0].n_uniform + (gplan.cls[0].extra ? 1 : 0);
    auto draw = [&](uint32_t t) {
      const StepUniform u = step_uniform(P, mu, t);
      uint64_t p0 = gplan.cls[0].p0;
#pragma unroll
      for (int e = 0; e < kPipeEvents; ++e) {
        if (e < n_mine) {
          uint32_t w0, w1, w2;
          philox_from_p0<true>(P, mu, u, p0, w0, w1, w2);
          dr_o[e] = __umulhi(w1, (uint32_t)P.noise_n);
          dr_q[e] = hi32((uint64_t)w2 * (uint32_t)P.noise_qmax + P.q_addend) | (w0 & 0x80000000u);
          p0 = add64_alu(p0, gplan.p0_inc.inc);
        }
      }
    };
    if (P.S > 0) draw(t0);
    for (long long s = 0; s < P.S; ++s) {
      const int4 ctl = *reinterpret_cast<const int4*>(s_ctl);
      last = ctl.x;
      RuleCtx rc;
      rc.last = last; rc.L = L; rc.dp = last - prev; rc.mid2 = 0; rc.mkt_flags = nullptr;
      rc.bid_lo = (uint32_t)ctl.y; rc.ask_lo = (uint32_t)ctl.z; rc.noclamp = ctl.w != 0;
      rc.bid_last = 0; rc.ask_last = 0;
      // a2: the orders drawn during the previous clearing go to their ticks
#pragma unroll
      for (int e = 0; e < kPipeEvents; ++e) {
        if (e < n_mine) {
          const uint32_t m = (uint32_t)((int32_t)dr_q[e] >> 31), o = dr_o[e];
          const int q = (int)(dr_q[e] & 0x7fffffffu);
          if (rc.noclamp) {
            const uint32_t bid_top = rc.bid_lo + (uint32_t)P.noise_n4;
            book_add_at<ATOM>(bref, (rc.ask_lo ^ (m & (rc.ask_lo ^ bid_top))) + ((o ^ m) << 2), q, sink);
          } else {
            const bool buy = m != 0u;
            const int tick = clamp_tick(buy ? (last + P.noise_delta) - (int)o : (last - P.noise_delta) + (int)o, L);
            book_add<ATOM>(bref, 4u * (uint32_t)(buy ? tick : tick + L), q, sink);
          }
        }
      }
      __syncthreads();                                   // B1: the combined book is complete
      if (warp == 0) clear_step(s, rc);                  // a3-a6 ...
      else if (s + 1 < P.S) draw(t0 + (uint32_t)s + 1u); // ... while the other warps draw the next step (a1)
      __syncthreads();                                   // B2: residual book and new price visible
      prev = last;
    }
  } else {
    for (long long s = 0; s < P.S; ++s) {
      const uint32_t t = t0 + (uint32_t)s;
      const StepUniform u = step_uniform(P, mu, t);
      const int4 ctl = *reinterpret_cast<const int4*>(s_ctl);
      last = ctl.x;
      RuleCtx rc;
      rc.last = last; rc.L = L;
      if constexpr (MODEL == 2) {
        rc.mid2 = ctl.y; rc.dp = ctl.z; rc.mkt_flags = s_mkt;
      {                                                // no-clamp path: midr +- dmax inside the grid
        const int midr = (rc.mid2 + 1) >> 1;
        rc.noclamp = midr - P.dmax >= 0 && midr + P.dmax <= L - 1;
        rc.bid_last = bref.saddr + 4u * (uint32_t)midr; rc.ask_last = rc.bid_last + 4u * (uint32_t)L;
        rc.bid_lo = rc.bid_last - 4u * (uint32_t)P.noise_delta; rc.ask_lo = rc.ask_last - 4u * (uint32_t)P.noise_delta;
      }
        generate_step_paper<ATOM>(P, bref, mu, u, rc, gplan, tid, t, sink);
      } else {
        rc.dp = last - prev; rc.mid2 = 0; rc.mkt_flags = nullptr;
        rc.bid_lo = (uint32_t)ctl.y; rc.ask_lo = (uint32_t)ctl.z; rc.noclamp = ctl.w != 0;
        rc.bid_last = rc.bid_lo + 4u * (uint32_t)P.noise_delta; rc.ask_last = rc.ask_lo + 4u * (uint32_t)P.noise_delta;
        // a1 + a2: order generation and aggregation
        generate_step<MODEL, ATOM, PACKED>(P, bref, mu, u, rc, gplan, tid == 0, sink);
      }
      __syncthreads();                                   // B1: the combined book is complete

      if (warp == 0) clear_step(s, rc);
      __syncthreads();                                   // B2: residual book and new price visible
      prev = last;
    }

  }

  // ---- a7: write-back (shared -> HBM), 16-byte vectors, plus the totals for sub_buy/sub_sell
  long long sb1 = 0, sa1 = 0;
  {
    const int nvec = L / 2, nside = L / 4;
    const int4* sbook4 = reinterpret_cast<const int4*>(book);
    int4* gbook4 = reinterpret_cast<int4*>(gbook);
    for (int i = tid; i < nvec; i += T) {
      int4 v = sbook4[i];
      gbook4[i] = v;
      long long sum = (long long)v.x + v.y + v.z + v.w;
      if (i < nside) sb1 += sum; else sa1 += sum;
    }
  }
  BookTotals tot1 = block_reduce_totals(sb1, sa1, -1, 0x7fffffff, s_red64, s_red32);
  if (tid == 0) {
    // submitted = (resting after - resting before) + executed during this run (conservation;
    // the oracle counts the same quantity order by order)
    long long dvol = s_rec[F_SUMVOL] - vol0;
    s_rec[F_SUBBUY] += (tot1.sum_bid - tot0.sum_bid) + dvol;
    s_rec[F_SUBSELL] += (tot1.sum_ask - tot0.sum_ask) + dvol;
    s_rec[F_NORDERS] += P.S * P.orders_per_step;
  }
  __syncthreads();
  if (tid < 16) grec[tid] = s_rec[tid];
}

// ks_create: empty books, opening price, zero accumulators (Alg.1 l.2-3).
__global__ void ks_init_kernel(int4* books4, size_t nvec, long long* recs, int M, int init_price, int init_prev) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  size_t stride = (size_t)gridDim.x * blockDim.x;
  for (size_t v = i; v < nvec; v += stride) books4[v] = make_int4(0, 0, 0, 0);
  for (size_t r = i; r < (size_t)M * 16; r += stride) {
    int f = (int)(r & 15);
    long long val = 0;
    if (f == F_LAST) val = init_price;
    if (f == F_PREV) val = init_prev;                  // model 4: the doubled opening price (previous mid)
    if (f == F_HASH) val = (long long)kHashBasis;
    recs[r] = val;
  }
}

// ks_write_books depth check: max over markets and sides of the total depth -> *out (atomicMax).
__global__ void ks_depth_bound_kernel(const int32_t* books, int L, unsigned long long* out) {
  const int32_t* side = books + (size_t)blockIdx.x * (size_t)L;      // grid = 2*M sides
  long long sum = 0; int neg = 0;
  for (int i = threadIdx.x; i < L; i += blockDim.x) { int v = side[i]; sum += v; neg |= (v < 0); }
  for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
  neg = __any_sync(0xffffffffu, neg);
  __shared__ long long s[32];
  __shared__ int sneg;
  if (threadIdx.x == 0) sneg = 0;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) { s[threadIdx.x >> 5] = sum; if (neg) sneg = 1; }
  __syncthreads();
  if (threadIdx.x == 0) {
    long long tot = 0;
    for (int w = 0; w < (int)((blockDim.x + 31) >> 5); ++w) tot += s[w];
    unsigned long long v = sneg ? 0xffffffffffffffffull : (unsigned long long)tot;
    atomicMax(out, v);
  }
}

}  // namespace ks
