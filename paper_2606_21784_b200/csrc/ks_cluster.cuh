// ks_cluster.cuh -- the persistent kernel for books that outgrow one SM's shared memory
// (north_star (2); the paper's "tiling" remark).  One thread-block CLUSTER per
// market: CTA rank r of a C-CTA cluster keeps ticks [r*Lc, (r+1)*Lc), Lc = L/C, of both sides in
// its own shared memory (book[2][Lc]); the cluster's C*T threads share the agents.  An order whose
// tick belongs to another CTA is added with a remote shared-memory reduction
// (red.shared::cluster over DSMEM); warp 0 of rank 0 clears the active window through
// ld/st.shared::cluster, so the clearing code is the one of ks_device.cuh with another accessor.
// Two cluster barriers per step replace the two __syncthreads() of the one-CTA kernel.
// Same definitions, same results, bit for bit (tests/test_gpu_parity.py runs both on one input).
#pragma once
#include "ks_kernel.cuh"

namespace ks {

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
// shared::cluster address of the same shared-memory location in CTA `rank` of this cluster
__device__ __forceinline__ uint32_t mapa_shared(uint32_t saddr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
  return r;
}
__device__ __forceinline__ void cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void st_cluster_s32(uint32_t caddr, int v) {
  asm volatile("st.shared::cluster.s32 [%0], %1;" ::"r"(caddr), "r"(v) : "memory");
}
__device__ __forceinline__ void st_cluster_s64(uint32_t caddr, long long v) {
  asm volatile("st.shared::cluster.s64 [%0], %1;" ::"r"(caddr), "l"(v) : "memory");
}

// Where tick `tick` of side `side` lives: CTA rank tick / Lc, word side*Lc + tick % Lc of its book.
struct ClusterBook {
  uint32_t saddr;        // shared-window address of this CTA's book (identical in every CTA)
  int log2Lc;
  __device__ __forceinline__ uint32_t addr(int side, int tick) const {
    const uint32_t rank = (uint32_t)tick >> log2Lc;
    const uint32_t loc = ((uint32_t)side << log2Lc) + ((uint32_t)tick & ((1u << log2Lc) - 1u));
    return mapa_shared(saddr + 4u * loc, rank);
  }
  __device__ __forceinline__ int4 ld4(int side, int tick) const {
    int4 v;
    asm volatile("ld.shared::cluster.v4.s32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr(side, tick)) : "memory");
    return v;
  }
  __device__ __forceinline__ void st4(int side, int tick, int4 v) const {
    asm volatile("st.shared::cluster.v4.s32 [%0], {%1, %2, %3, %4};"
                 ::"r"(addr(side, tick)), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
  }
  __device__ __forceinline__ int ld1(int side, int tick) const {
    int v;
    asm volatile("ld.shared::cluster.s32 %0, [%1];" : "=r"(v) : "r"(addr(side, tick)) : "memory");
    return v;
  }
  __device__ __forceinline__ void st1(int side, int tick, int v) const { st_cluster_s32(addr(side, tick), v); }
};

// grid = M*C CTAs in clusters of C = 1 << P.log2C (cluster <-> market), block = T threads,
// dynamic shared memory = 8*Lc bytes.  MODEL: 0 = ZI, 1 = MIX3.
template <int MODEL, bool PACKED>
__global__ void __launch_bounds__(1024, 1) ks_cluster_kernel(const __grid_constant__ KernelParams P) {
  extern __shared__ __align__(16) int32_t book[];     // [2][Lc]: this CTA's ticks, bid then ask
  __shared__ long long s_rec[16];
  __shared__ long long s_red64[64];
  __shared__ int s_red32[64];
  __shared__ int2 s_trace[32];                        // staged trace entries (rank 0, only when P.trace)
  __shared__ int s_ctl[4];                            // [0] = price at the start of the step (written by rank 0)
  __shared__ long long s_ctot[8][2];                  // rank 0 only: per-rank (sum_bid, sum_ask)
  __shared__ int s_cext[8][2];                        // rank 0 only: per-rank (bmax, amin), global ticks
  __shared__ int s_abort;
  __shared__ int s_ovf;

  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5;
  const int L = P.L, log2C = P.log2C, C = 1 << log2C;
  int log2L = 0;
  while ((1 << log2L) < L) ++log2L;
  const int log2Lc = log2L - log2C, Lc = 1 << log2Lc;
  const uint32_t rank = cluster_ctarank();
  const uint32_t cluster_id = blockIdx.x >> log2C;
  const uint32_t market = P.market_base + cluster_id;
  int32_t* gbook = P.books + (size_t)cluster_id * 2 * (size_t)L;
  long long* grec = P.recs + (size_t)cluster_id * 16;
  const MarketUniform mu = market_uniform(P, market);
  const GenPlan<MODEL> gplan = gen_plan<MODEL>(PACKED ? (uint32_t)P.A >> 2 : (uint32_t)P.A, (int)rank * T + tid, C * T);
  BookRef bref; bref.ptr = book; bref.saddr = (uint32_t)__cvta_generic_to_shared(book);
  bref.log2L = log2L; bref.log2Lc = log2Lc;
  const ClusterBook io{bref.saddr, log2Lc};
  const uint32_t ctl_saddr = (uint32_t)__cvta_generic_to_shared(s_ctl);
  const uint32_t ctot_saddr = (uint32_t)__cvta_generic_to_shared(&s_ctot[rank][0]);
  const uint32_t cext_saddr = (uint32_t)__cvta_generic_to_shared(&s_cext[rank][0]);
  const int tick_base = (int)rank * Lc;

  // deferred depth check of ks_write_books (as in ks_persistent_kernel): a uniform decision of the
  // whole grid, taken before any cluster barrier
  if (P.depth_word) {
    if (tid == 0) {
      const unsigned long long b = *P.depth_word;
      s_abort = b > P.depth_limit;
      if (b > P.depth_limit && blockIdx.x == 0) {
        *P.host_flags = b == 0xffffffffffffffffull ? kFlagNegativeDepth : kFlagDepthOverflow;
        __threadfence_system();
      }
    }
    __syncthreads();
    if (s_abort) return;
  }
  // every CTA of the cluster must be running before its shared memory is written remotely
  cluster_sync();

  // ---- a0: every CTA loads its own ticks
  long long sb0 = 0, sa0 = 0;
  int bmax = -1, amin = 0x7fffffff;
  {
    const int nside = Lc / 4;
    int4* sbook4 = reinterpret_cast<int4*>(book);
    if (P.fresh) {
      for (int i = tid; i < 2 * nside; i += T) sbook4[i] = make_int4(0, 0, 0, 0);
    } else {
      const int4* gbid4 = reinterpret_cast<const int4*>(gbook + tick_base);
      const int4* gask4 = reinterpret_cast<const int4*>(gbook + L + tick_base);
      for (int i = tid; i < 2 * nside; i += T) {
        const bool is_bid = i < nside;
        const int j0 = is_bid ? i : i - nside;
        int4 v = __ldg((is_bid ? gbid4 : gask4) + j0);
        sbook4[i] = v;
        int vals[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const int tick = tick_base + 4 * j0 + j;
          if (is_bid) { sb0 += vals[j]; if (vals[j] > 0) bmax = max(bmax, tick); }
          else        { sa0 += vals[j]; if (vals[j] > 0) amin = min(amin, tick); }
        }
      }
    }
    if (tid < 16) s_rec[tid] = grec[tid];
  }
  BookTotals tot0 = block_reduce_totals(sb0, sa0, bmax, amin, s_red64, s_red32);   // has barriers
  if (tid == 0) {
    st_cluster_s64(mapa_shared(ctot_saddr, 0), tot0.sum_bid);
    st_cluster_s64(mapa_shared(ctot_saddr + 8, 0), tot0.sum_ask);
    st_cluster_s32(mapa_shared(cext_saddr, 0), tot0.bmax);
    st_cluster_s32(mapa_shared(cext_saddr + 4, 0), tot0.amin);
  }
  int last = (int)s_rec[F_LAST], prev = (int)s_rec[F_PREV];
  const uint32_t t0 = (uint32_t)s_rec[F_STEPS];
  const long long vol0 = s_rec[F_SUMVOL];
  if (tid == 0) { s_ctl[0] = last; s_ovf = 0; }
  cluster_sync();
  long long tot0_bid = 0, tot0_ask = 0;
  bmax = -1; amin = L;
  if (rank == 0) {
    for (int r = 0; r < C; ++r) {
      tot0_bid += s_ctot[r][0]; tot0_ask += s_ctot[r][1];
      bmax = max(bmax, s_cext[r][0]); amin = min(amin, s_cext[r][1]);
    }
  }

  int sink = 0;
  // ---- S steps, all on-chip
  for (long long s = 0; s < P.S; ++s) {
    const uint32_t t = t0 + (uint32_t)s;
    const StepUniform u = step_uniform(P, mu, t);
    last = s_ctl[0];
    RuleCtx rc;
    rc.last = last; rc.dp = last - prev; rc.L = L; rc.noclamp = false; rc.bid_lo = 0; rc.ask_lo = 0;
    generate_step<MODEL, 3, PACKED>(P, bref, mu, u, rc, gplan, rank == 0 && tid == 0, sink);
    cluster_sync();                                    // B1: the combined book is complete in every CTA

    if (rank == 0 && warp == 0) {
      int lo = max(0, min(amin, last - P.dmax));
      int hi = min(L - 1, max(bmax, last + P.dmax));
      int vmax, pstar, nb, na, base, wend;
      LaneBounds lbnd;
      int width4 = hi - (lo & ~3) + 1, width8 = hi - (lo & ~7) + 1;
      if (P.force_generic || width8 > 256) { base = lo & ~3; wend = min(L, hi + 1); clear_generic(io, L, base, hi, lane, vmax, pstar, lbnd); }
      else if (hi - lo < 32)               { base = lo; wend = min(L, base + 32); clear_rows<1>(io, L, base, lane, vmax, pstar, lbnd); }
      else if (width4 <= 128)              { base = lo & ~3; wend = min(L, base + 128); clear_window<4>(io, L, base, lane, vmax, pstar, lbnd); }
      else                                 { base = lo & ~7; wend = min(L, base + 256); clear_window<8>(io, L, base, lane, vmax, pstar, lbnd); }
      reduce_bounds(lbnd, base, wend, nb, na);
      bmax = nb; amin = na;
      if (lane < C) st_cluster_s32(mapa_shared(ctl_saddr, (uint32_t)lane), vmax > 0 ? pstar : last);
      update_record_lanes(s_rec, &s_ovf, lane, last, vmax, pstar, last);
      if (P.trace) trace_step(s_trace, P.trace + (size_t)cluster_id * (size_t)P.S, s, P.S, lane,
                              vmax > 0 ? pstar : last, vmax);
    }
    cluster_sync();                                    // B2: residual book and new price visible
    prev = last;
  }

  // ---- a7: every CTA writes its own ticks back; totals go to rank 0
  long long sb1 = 0, sa1 = 0;
  {
    const int nside = Lc / 4;
    const int4* sbook4 = reinterpret_cast<const int4*>(book);
    int4* gbid4 = reinterpret_cast<int4*>(gbook + tick_base);
    int4* gask4 = reinterpret_cast<int4*>(gbook + L + tick_base);
    for (int i = tid; i < 2 * nside; i += T) {
      int4 v = sbook4[i];
      long long sum = (long long)v.x + v.y + v.z + v.w;
      if (i < nside) { gbid4[i] = v; sb1 += sum; } else { gask4[i - nside] = v; sa1 += sum; }
    }
  }
  BookTotals tot1 = block_reduce_totals(sb1, sa1, -1, 0x7fffffff, s_red64, s_red32);
  if (tid == 0) {
    st_cluster_s64(mapa_shared(ctot_saddr, 0), tot1.sum_bid);
    st_cluster_s64(mapa_shared(ctot_saddr + 8, 0), tot1.sum_ask);
  }
  cluster_sync();
  if (rank == 0) {
    if (tid == 0) {
      long long tot1_bid = 0, tot1_ask = 0;
      for (int r = 0; r < C; ++r) { tot1_bid += s_ctot[r][0]; tot1_ask += s_ctot[r][1]; }
      long long dvol = s_rec[F_SUMVOL] - vol0;
      s_rec[F_SUBBUY] += (tot1_bid - tot0_bid) + dvol;
      s_rec[F_SUBSELL] += (tot1_ask - tot0_ask) + dvol;
      s_rec[F_NORDERS] += P.S * P.orders_per_step;
      if (s_ovf) { *P.host_flags = kFlagStatOverflow; __threadfence_system(); }
    }
    __syncthreads();
    if (tid < 16) grec[tid] = s_rec[tid];
  }
  if (sink == 0x7fffffff) grec[0] = 0;                 // never taken (sink is unused here)
}

}  // namespace ks
