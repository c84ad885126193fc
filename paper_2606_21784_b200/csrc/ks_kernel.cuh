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

// a6: price state, statistics and trajectory hash -- all sixteen fields of the record
// (include/kineticsim.h, ks_market_stats) updated IN PARALLEL, lane f (f < 16) of the clearing warp
// owning field f: one LDS.64, a handful of warp instructions with a dependency depth of ~8, one
// STS.64 -- instead of fifteen dependent read-modify-writes by one lane.  The record stays in
// shared memory between steps (holding it in registers across the generation loop costs that
// loop four registers of its 64 and measured 2-7 % slower on C4 / C5).  Every additive field's
// per-step increment is a product X*Y of two of {0, 1, traded, Vmax, pt, r, r^2} (pt = p* on a
// trading step, else 0; r = last_after - last_before):
//   steps 1*1   n_trades 1*traded   sum_vol 1*Vmax   sum_px 1*pt   sum_px2 pt*pt   sum_pxvol pt*Vmax
//   sum_ret 1*r   sum_ret2 r*r   sum_ret3 r*r^2   sum_ret4 r^2*r^2   (others 0*0)
// so a lane picks its two factors by a constant 3-bit code and does ONE 32x32->64 multiply-add.
// f[12] last, f[13] prev and f[14] the trajectory hash are set, not added.  Signed overflow of any
// additive field (only sum_ret3 / sum_ret4 can get there: (L-1)^4 * steps may pass 2^63 on a wide
// grid) is detected exactly and raised as a sticky flag (KS_ERR_OVERFLOW, ks_api.cu).
__device__ __forceinline__ int rec_pick(int code, int tr, int vmax, int pt, int r, int r2) {
  // code: 0 zero, 1 one, 2 traded, 3 Vmax, 4 pt, 5 r, 6 r^2
  const bool b0 = code & 1, b1 = code & 2, b2 = code & 4;
  const int v01 = b0 ? 1 : 0, v23 = b0 ? vmax : tr, v45 = b0 ? r : pt;
  const int lo = b1 ? v23 : v01, hi = b1 ? r2 : v45;
  return b2 ? hi : lo;
}

// One step's record update by all lanes of the clearing warp.  prev_value is what f[13] receives
// (the price before the step; model 4: the doubled mid the step started from).  *ovf_flag (shared)
// is set when an additive field leaves int64.
__device__ __forceinline__ void update_record_lanes(long long* rec, int* ovf_flag, int lane, int last, int vmax, int pstar,
                                                    int prev_value) {
  //                         field: 15 14 13 12 11 10  9  8  7  6  5  4  3  2  1  0
  const unsigned long long XC = 0x0000006551441111ull;
  const unsigned long long YC = 0x0000006655344321ull;
  const int f = lane & 15;
  const int xc = (int)((XC >> (4 * f)) & 7ull), yc = (int)((YC >> (4 * f)) & 7ull);
  const int tr = vmax > 0 ? 1 : 0;
  const int new_last = tr ? pstar : last;
  const int pt = tr ? pstar : 0;
  const int r = new_last - last, r2 = r * r;            // |r| < 2^15, r^2 < 2^30
  const long long old = rec[f];
  const long long inc = (long long)rec_pick(xc, tr, vmax, pt, r, r2) * (long long)rec_pick(yc, tr, vmax, pt, r, r2);
  const long long sum = (long long)((unsigned long long)old + (unsigned long long)inc);
  const unsigned long long x = tr ? (((unsigned long long)(unsigned)vmax << 16) | (unsigned long long)(unsigned)pstar) : 0xFFFFull;
  const long long hash = (long long)(((unsigned long long)old ^ x) * kHashPrime);
  const long long nv = f == F_HASH ? hash : (f == F_LAST ? (long long)new_last : (f == F_PREV ? (long long)prev_value : sum));
  if (lane < 16) {
    rec[f] = nv;
    if (((old ^ sum) & (inc ^ sum)) < 0) *ovf_flag = 1;  // both operands of one sign, the sum of the other
  }
}

// The same update with the lane's field held in a REGISTER (ks_decoupled_kernel's bookkeeping warp:
// no shared-memory round trip per step); ovf is a per-lane sticky flag.
__device__ __forceinline__ void update_record_reg(long long& rec, int& ovf, int lane, int last, int vmax, int pstar,
                                                  int prev_value) {
  const unsigned long long XC = 0x0000006551441111ull;
  const unsigned long long YC = 0x0000006655344321ull;
  const int f = lane & 15;
  const int xc = (int)((XC >> (4 * f)) & 7ull), yc = (int)((YC >> (4 * f)) & 7ull);
  const int tr = vmax > 0 ? 1 : 0;
  const int new_last = tr ? pstar : last;
  const int pt = tr ? pstar : 0;
  const int r = new_last - last, r2 = r * r;
  const long long old = rec;
  const long long inc = (long long)rec_pick(xc, tr, vmax, pt, r, r2) * (long long)rec_pick(yc, tr, vmax, pt, r, r2);
  const long long sum = (long long)((unsigned long long)old + (unsigned long long)inc);
  const unsigned long long x = tr ? (((unsigned long long)(unsigned)vmax << 16) | (unsigned long long)(unsigned)pstar) : 0xFFFFull;
  const long long hash = (long long)(((unsigned long long)old ^ x) * kHashPrime);
  rec = f == F_HASH ? hash : (f == F_LAST ? (long long)new_last : (f == F_PREV ? (long long)prev_value : sum));
  if (((old ^ sum) & (inc ^ sum)) < 0) ovf = 1;          // inc = 0 for the fields that are set, not added
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

__device__ __forceinline__ int sign_of(int x) { return (x > 0) - (x < 0); }

// Split-phase named barriers (PTX bar.arrive / bar.sync on barrier `id`, `n` participating
// threads): the producer side of a phase only ARRIVES and goes on, the consumer side waits
// (producer/consumer use as in the PTX ISA's bar.arrive example).  Used by ks_decoupled_kernel
// only: inside ks_persistent_kernel's step loop they sit in a branch the compiler must treat as
// divergent, and ptxas then stops keeping the Philox keys in uniform registers across the
// generation loops (measured: +5 % instructions on C5) -- that kernel keeps __syncthreads().
// The barrier id is an immediate: with an id in a register ptxas reserves all 16 hardware barriers
// for the CTA (4 resident CTAs per SM at most).
template <int ID> __device__ __forceinline__ void bar_sync(int n) { asm volatile("bar.sync %0, %1;" ::"n"(ID), "r"(n) : "memory"); }
template <int ID> __device__ __forceinline__ void bar_arrive(int n) { asm volatile("bar.arrive %0, %1;" ::"n"(ID), "r"(n) : "memory"); }

// ---- pieces shared by the kernels of this file ------------------------------------------------
// Deferred depth check of ks_write_books (ks_api.cu): every CTA reads the same device word and
// takes the same decision, so an unsafe run changes nothing at all.  Returns true = abort.
__device__ __forceinline__ bool depth_check_aborts(const KernelParams& P, int* s_abort) {
  if (!P.depth_word) return false;
  if (threadIdx.x == 0) {
    const unsigned long long b = *P.depth_word;
    *s_abort = b > P.depth_limit;
    if (b > P.depth_limit && blockIdx.x == 0) {
      *P.host_flags = b == 0xffffffffffffffffull ? kFlagNegativeDepth : kFlagDepthOverflow;
      __threadfence_system();
    }
  }
  __syncthreads();
  return *s_abort != 0;
}

// Bulk asynchronous copies (TMA engine, no tensor map): ONE elected thread moves a whole 8*L-byte
// book between HBM and shared memory, so the state phase does not depend on how many threads the
// CTA has (32 for the throughput plan: 32 threads of int4 loads left the copy engine idle) and the
// other threads hold no registers or LSU slots for it.  Sizes are multiples of 16 bytes (L >= 32),
// both addresses 16-byte aligned (d_state is, and 8*L is a multiple of 256).
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(done) : "r"(mbar), "r"(parity) : "memory");
  } while (!done);
}
__device__ __forceinline__ void bulk_load(uint32_t dst_smem, const void* src_gmem, uint32_t bytes, uint32_t mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst_smem), "l"(src_gmem), "r"(bytes), "r"(mbar) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dst_gmem, uint32_t src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(src_smem), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
// the bulk stores of this thread have READ their shared-memory source (the CTA may exit)
__device__ __forceinline__ void bulk_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// generic-proxy writes of this thread to shared memory become visible to the async proxy (the copy engine)
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// a0: state load (HBM -> shared) of one market's [2][L] book, skipped for a fresh (all-zero) book:
// one bulk copy of 8*L bytes issued by thread 0, completion on an mbarrier every thread waits on;
// then a pass over SHARED memory gives the per-thread partial depth totals and extents of what was
// loaded.
__device__ __forceinline__ void load_book(const KernelParams& P, int32_t* book, const int32_t* gbook, int L,
                                          long long& sb0, long long& sa0, int& bmax, int& amin) {
  const int tid = threadIdx.x, T = blockDim.x;
  const int nvec = L / 2;                              // int4 vectors in the whole book
  int4* sbook4 = reinterpret_cast<int4*>(book);
  sb0 = 0; sa0 = 0; bmax = -1; amin = 0x7fffffff;
  if (P.fresh) {
    for (int i = tid; i < nvec; i += T) sbook4[i] = make_int4(0, 0, 0, 0);
  } else {
    __shared__ __align__(8) unsigned long long s_load_mbar;
    const uint32_t mbar = (uint32_t)__cvta_generic_to_shared(&s_load_mbar);
    if (tid == 0) {
      mbar_init(mbar, 1);
      mbar_expect_tx(mbar, 8u * (uint32_t)L);
      bulk_load((uint32_t)__cvta_generic_to_shared(book), gbook, 8u * (uint32_t)L, mbar);
    }
    __syncthreads();                                   // the barrier object exists before anybody polls it
    mbar_wait(mbar, 0);
    // Depths are >= 0 and a side's total stays below 2^31 (the guards of ks_run; ks_write_books and
    // ks_attach refuse negative entries), so a thread's partial sums fit 32 bits and "this vector
    // holds depth" is "its sum is not zero".  Per 16-byte vector: one LDS.128, the sum, one compare;
    // the tick inside the extreme vector is found once, after the loops (with 32 threads and 4 KB of
    // book the state phase is bound by instruction issue, not by HBM: profiles/r3_state_io.md).
    const int nside = L / 4;
    int s32b = 0, s32a = 0, ib = -1, ia = -1;
    for (int i = tid; i < nside; i += T) {             // bids: the LAST vector with depth (i increases)
      const int4 v = sbook4[i];
      const int sum = (v.x + v.y) + (v.z + v.w);
      s32b += sum;
      ib = sum != 0 ? i : ib;
    }
    for (int i = nside + tid; i < nvec; i += T) {      // asks: the FIRST vector with depth
      const int4 v = sbook4[i];
      const int sum = (v.x + v.y) + (v.z + v.w);
      s32a += sum;
      ia = (sum != 0 && ia < 0) ? i : ia;
    }
    sb0 = s32b; sa0 = s32a;
    if (ib >= 0) { const int4 v = sbook4[ib]; bmax = 4 * ib + (v.w > 0 ? 3 : v.z > 0 ? 2 : v.y > 0 ? 1 : 0); }
    if (ia >= 0) { const int4 v = sbook4[ia]; amin = 4 * (ia - nside) + (v.x > 0 ? 0 : v.y > 0 ? 1 : v.z > 0 ? 2 : 3); }
  }
}

// a7: write-back (shared -> HBM) of the book with ONE bulk copy and of the 128-byte record; the
// depth totals (a pass over shared memory) give sub_buy / sub_sell by conservation: submitted =
// (resting after - resting before) + executed during this run (the oracle counts the same quantity
// order by order).  keep[3] = resting bid total, resting ask total, executed volume at the start
// of the run.  Every thread fences its own book writes towards the copy engine before the barriers
// of the reduction; thread 0 issues the copy after them and keeps the CTA alive until the engine
// has read the book.
__device__ __forceinline__ void store_state(const KernelParams& P, const int32_t* book, int32_t* gbook, long long* grec, int L,
                                            long long* s_rec, const long long* keep, const int* s_ovf,
                                            long long* s_red64, int* s_red32) {
  const int tid = threadIdx.x, T = blockDim.x;
  int s32b = 0, s32a = 0;                              // 32 bits suffice: see load_book
  fence_proxy_async_smem();
  {
    const int nvec = L / 2, nside = L / 4;
    const int4* sbook4 = reinterpret_cast<const int4*>(book);
    for (int i = tid; i < nside; i += T) { const int4 v = sbook4[i]; s32b += (v.x + v.y) + (v.z + v.w); }
    for (int i = nside + tid; i < nvec; i += T) { const int4 v = sbook4[i]; s32a += (v.x + v.y) + (v.z + v.w); }
  }
  BookTotals tot1 = block_reduce_totals((long long)s32b, (long long)s32a, -1, 0x7fffffff, s_red64, s_red32);     // has barriers
  if (tid == 0) {
    bulk_store(gbook, (uint32_t)__cvta_generic_to_shared(book), 8u * (uint32_t)L);
    long long dvol = s_rec[F_SUMVOL] - keep[2];
    s_rec[F_SUBBUY] += (tot1.sum_bid - keep[0]) + dvol;
    s_rec[F_SUBSELL] += (tot1.sum_ask - keep[1]) + dvol;
    s_rec[F_NORDERS] += P.S * P.orders_per_step;
    if (*s_ovf) { *P.host_flags = kFlagStatOverflow; __threadfence_system(); }
  }
  __syncthreads();
  if (tid < 16) grec[tid] = s_rec[tid];
  if (tid == 0) bulk_store_wait_read();
}

// a3-a5 on the active window [lo, hi] of a book in this CTA's shared memory, by one warp: picks
// the scan by the window's width.  base / wend = the tick range the chosen scan covered.
__device__ __forceinline__ void clear_active_window(const LocalBook& io, int L, int lo, int hi, bool force_generic, int lane,
                                                    int& vmax, int& pstar, LaneBounds& lbnd, int& base, int& wend) {
  const int width4 = hi - (lo & ~3) + 1, width8 = hi - (lo & ~7) + 1;
  if (force_generic || width8 > 256) { base = lo & ~3; wend = min(L, hi + 1); clear_generic(io, L, base, hi, lane, vmax, pstar, lbnd); }
  else if (hi - lo < 32)             { base = lo; wend = min(L, base + 32); clear_rows<1>(io, L, base, lane, vmax, pstar, lbnd); }
  else if (hi - lo < 64)             { base = lo; wend = min(L, base + 64); clear_rows<2>(io, L, base, lane, vmax, pstar, lbnd); }
  else if (width4 <= 128)            { base = lo & ~3; wend = min(L, base + 128); clear_window<4>(io, L, base, lane, vmax, pstar, lbnd); }
  else                               { base = lo & ~7; wend = min(L, base + 256); clear_window<8>(io, L, base, lane, vmax, pstar, lbnd); }
}

// Model 4: the same on the window the limit orders span, with the step's marketable depth at the
// grid's edge ticks (bid[L-1], ask[0]) counted as ExtDepth when the chosen scan does not reach
// them -- so that a marketable order does not turn the step into a full-grid scan.  Returns false,
// having written nothing, when the exactness condition of ExtDepth fails or the window needs the
// chunked scan; the caller then scans to the edge.  On success the edge ticks end empty.
__device__ __forceinline__ bool clear_active_window_ext(const LocalBook& io, int L, int lo, int hi, bool mkt_buy, bool mkt_sell,
                                                        int lane, int& vmax, int& pstar, LaneBounds& lbnd, int& base, int& wend) {
  const int width4 = hi - (lo & ~3) + 1, width8 = hi - (lo & ~7) + 1;
  int path;
  if (width8 > 256)       return false;
  else if (hi - lo < 32)  { path = 1; base = lo; wend = min(L, base + 32); }
  else if (hi - lo < 64)  { path = 2; base = lo; wend = min(L, base + 64); }
  else if (width4 <= 128) { path = 4; base = lo & ~3; wend = min(L, base + 128); }
  else                    { path = 8; base = lo & ~7; wend = min(L, base + 256); }
  ExtDepth ext;
  ext.b = (mkt_buy && wend <= L - 1) ? io.ld1(0, L - 1) : 0;    // a scan that reaches the edge tick counts it itself
  ext.a = (mkt_sell && base > 0) ? io.ld1(1, 0) : 0;
  bool ok;
  if (path == 1)      ok = clear_rows<1, LocalBook, false, true>(io, L, base, lane, vmax, pstar, lbnd, nullptr, nullptr, ext);
  else if (path == 2) ok = clear_rows<2, LocalBook, false, true>(io, L, base, lane, vmax, pstar, lbnd, nullptr, nullptr, ext);
  else if (path == 4) ok = clear_window<4, LocalBook, false, true>(io, L, base, lane, vmax, pstar, lbnd, nullptr, nullptr, ext);
  else                ok = clear_window<8, LocalBook, false, true>(io, L, base, lane, vmax, pstar, lbnd, nullptr, nullptr, ext);
  if (ok && lane == 0) {
    if (ext.b != 0) io.st1(0, L - 1, 0);
    if (ext.a != 0) io.st1(1, 0, 0);
  }
  __syncwarp();
  return ok;
}

// ---------------------------------------------------------------------------------------------
// The persistent kernel.  grid = M CTAs (one per market), block = T threads (any multiple of 32),
// dynamic shared memory = 8*L bytes (the book).  MODEL: 0 = ZI, 1 = MIX3, 2 = the paper's agent
// model (mid-price reference, A24).  ATOM: see book_add.
// PACKED: the PACKED4 draw contract (one Philox block per four agents, A22).
//
// Step structure (Alg.1 phases): a1+a2 by all warps | barrier | a3-a6 by ONE
// clearing warp | barrier.  The clearing warp is warp (blockIdx mod #warps): warps map to the SM's
// four schedulers by index, so a fixed warp 0 would pile every resident market's clearing on one
// scheduler.  This is the throughput kernel (many markets per SM hide each other's clearing; the
// automatic plan runs it with ONE warp per market on C4); when the grid underfills the GPU the
// step latency counts and ks_decoupled_kernel takes over.
// ---------------------------------------------------------------------------------------------
template <int MODEL, int ATOM, bool PACKED>
__global__ void __launch_bounds__(1024, 1) ks_persistent_kernel(const __grid_constant__ KernelParams P) {
  extern __shared__ __align__(16) int32_t book[];     // [2][L]: bid then ask
  __shared__ long long s_rec[16];
  __shared__ long long s_red64[64];
  __shared__ int s_red32[64];
  __shared__ int2 s_trace[32];                        // staged trace entries (only when P.trace)
  __shared__ __align__(16) int s_ctl[4];              // per-step broadcast: last, &bid[last-delta], &ask[last-delta], noclamp
                                                      // (MODEL 2: last, mid2, sgn(mid2 - previous mid2), 0)
  __shared__ int s_mkt[2];                            // MODEL 2: a marketable buy / sell was generated this step
  __shared__ int s_abort;
  __shared__ int s_ovf;                               // an int64 statistic overflowed (sticky)
  __shared__ long long s_keep[3];                     // resting totals and executed volume at the start of the run:
                                                      // parked here so that they hold no registers during the S steps

  const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5;
  const int L = P.L;
  const bool clearing = warp == (int)(blockIdx.x % (unsigned)(T >> 5));   // the clearing warp of this market
  const uint32_t market = P.market_base + blockIdx.x;
  int32_t* gbook = P.books + (size_t)blockIdx.x * 2 * (size_t)L;
  long long* grec = P.recs + (size_t)blockIdx.x * 16;
  if (depth_check_aborts(P, &s_abort)) return;
  const MarketUniform mu = market_uniform(P, market);
  const GenPlan<MODEL> gplan = make_gen_plan<MODEL>(P, PACKED, tid, T);
  BookRef bref; bref.ptr = book; bref.saddr = (uint32_t)__cvta_generic_to_shared(book);
#ifdef KS_DEBUG_CHECKS
  __shared__ int s_dbg_count;
  bref.dbg_lo = bref.saddr; bref.dbg_hi = bref.saddr + 8u * (uint32_t)L; bref.dbg_count = &s_dbg_count;
  if (tid == 0) s_dbg_count = 0;
#endif

  // ---- a0
  long long sb0, sa0;
  int bmax, amin;
  load_book(P, book, gbook, L, sb0, sa0, bmax, amin);
  if (tid < 16) s_rec[tid] = grec[tid];
  if (tid == 0) s_ovf = 0;
  BookTotals tot0 = block_reduce_totals(sb0, sa0, bmax, amin, s_red64, s_red32);   // has barriers
  bmax = tot0.bmax;                       // only the clearing warp keeps these up to date below
  amin = min(tot0.amin, L);
  int last = (int)s_rec[F_LAST], prev = (int)s_rec[F_PREV];
  const uint32_t t0 = (uint32_t)s_rec[F_STEPS];
  const uint32_t S = (uint32_t)P.S;                   // ks_run guarantees steps_done + S < 2^32
  if (tid == 0) { s_keep[0] = tot0.sum_bid; s_keep[1] = tot0.sum_ask; s_keep[2] = s_rec[F_SUMVOL]; }

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
  // a3-a6: clearing by the clearing warp on the active window
  auto clear_step = [&](uint32_t s, int mid2_now) {
#ifdef KS_DEBUG_CHECKS
    // B1 held: exactly this step's orders are in the book, and none of the next step's yet
    if (lane == 0) { KS_CHECK((long long)s_dbg_count == P.orders_per_step, "orders in the book at B1 != orders of the step"); s_dbg_count = 0; }
    __syncwarp();
#endif
    int lo, hi;
    int vmax, pstar, base, wend, nb, na;
    LaneBounds lbnd;
    const LocalBook io{book, L};
    bool cleared = false;
    if (MODEL == 2) {
      lo = max(0, min(amin, (mid2_now >> 1) - P.dmax));
      hi = min(L - 1, max(bmax, ((mid2_now + 1) >> 1) + P.dmax));
      const bool mkt_buy = s_mkt[0] != 0, mkt_sell = s_mkt[1] != 0;   // marketable buys sit at tick L-1, sells at tick 0
      __syncwarp();
      if ((mkt_buy || mkt_sell) && !P.force_generic)
        cleared = clear_active_window_ext(io, L, lo, hi, mkt_buy, mkt_sell, lane, vmax, pstar, lbnd, base, wend);
      if (!cleared) {                                // the scan reaches the edge ticks itself
        if (mkt_buy) hi = L - 1;
        if (mkt_sell) lo = 0;
      }
    } else {
      lo = max(0, min(amin, last - P.dmax));
      hi = min(L - 1, max(bmax, last + P.dmax));
    }
    if (!cleared) clear_active_window(io, L, lo, hi, P.force_generic != 0, lane, vmax, pstar, lbnd, base, wend);
    reduce_bounds(lbnd, base, wend, nb, na);
    if (MODEL == 2) {
      // the mid price needs the EXACT best quotes: a side with no depth inside the window is
      // searched outside it (rare: the window was emptied on that side)
      if (nb < base) nb = best_bid_below(io, L, base, lane);
      if (na >= wend) na = best_ask_from(io, L, wend, lane);
      if (lane == 0) { publish_paper(vmax > 0 ? pstar : last, nb, na, mid2_now); s_mkt[0] = 0; s_mkt[1] = 0; }
    } else {
      if (lane == 0) publish(vmax > 0 ? pstar : last);
    }
    bmax = nb; amin = na;
    update_record_lanes(s_rec, &s_ovf, lane, last, vmax, pstar, MODEL == 2 ? mid2_now : last);
    if (P.trace) trace_step(s_trace, P.trace + (size_t)blockIdx.x * (size_t)S, (long long)s, (long long)S, lane,
                            vmax > 0 ? pstar : last, vmax);
  };
  // ---- S steps, all on-chip
  for (uint32_t s = 0; s < S; ++s) {
    const uint32_t t = t0 + s;
#ifdef KS_DEBUG_INJECT_RACE                            // negative control: B1 dropped and the other warps made late
    if (!clearing) __nanosleep(20000);
#endif
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
#ifndef KS_DEBUG_INJECT_RACE                           // (the negative control of the KS_DEBUG_CHECKS build drops B1)
    __syncthreads();                                   // B1: the combined book is complete
#endif
    if (clearing) clear_step(s, rc.mid2);
    __syncthreads();                                   // B2: residual book and new price visible
    prev = last;
  }

  // ---- a7
  store_state(P, book, gbook, grec, L, s_rec, s_keep, &s_ovf, s_red64, s_red32);
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

// ks_attach record check: out[0] = max over markets of the step counter f[0] (atomicMax), out[1] = 1
// when some record could not have been written by this library: f[0] < 0, last (f[12]) outside
// [0, L), or f[13] outside [0, prev_limit) -- prev_limit = L for a previous price, 2L-1 for the
// doubled mid of KS_MODEL_PAPER.  Such prices would reach the rules' tick arithmetic unclamped.
__global__ void ks_attach_check_kernel(const long long* recs, int M, int L, int prev_limit, unsigned long long* out) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  long long steps = 0; int bad = 0;
  if (m < M) {
    const long long* r = recs + (size_t)m * 16;
    steps = r[F_STEPS];
    const long long last = r[F_LAST], prev = r[F_PREV];
    bad = steps < 0 || last < 0 || last >= L || prev < 0 || prev >= prev_limit;
    if (steps < 0) steps = 0;
  }
  for (int d = 16; d > 0; d >>= 1) { const long long o = __shfl_xor_sync(0xffffffffu, steps, d); steps = o > steps ? o : steps; }
  bad = __any_sync(0xffffffffu, bad);
  if ((threadIdx.x & 31) == 0) {
    atomicMax(out, (unsigned long long)steps);
    if (bad) out[1] = 1ull;
  }
}

}  // namespace ks
