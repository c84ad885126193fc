// ks_device.cuh -- device side of the call-auction clearing library (sm_100a).
//
// One CTA per market.  The int32 book (bid[L], ask[L]) lives in shared memory for all S steps
// (Alg.1).  Per step: every thread generates orders for its agents with
// Philox4x32-10 and adds them to the book with shared-memory atomics (a1, a2); one warp then
// clears the ACTIVE WINDOW of the book with a warp-shuffle scan (a3-a5) and updates the price
// state and the int64 statistics (a6).  Two __syncthreads() per step in ks_persistent_kernel
// (ks_kernel.cuh); in ks_decoupled_kernel (ks_decoupled.cuh) generation runs ahead of the clearing
// through a ring of price-independent histograms; ks_cluster_kernel (ks_cluster.cuh) splits a book
// over the CTAs of a cluster.  This file holds what they share: Philox, the agent rules, the
// aggregation and the clearing scans.
//
// tests/test_window_arguments.py checks the two exactness arguments used below (the window, and
// ExtDepth) by brute force against the full-grid definition.
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
#include <cstdio>
#include <cuda_runtime.h>

#ifndef KS_GEN_UNROLL
#define KS_GEN_UNROLL 4      // independent Philox chains per thread in the generation loop (measured on C4:
#endif                       // x2 404, x3 407, x4 409 G events/s); PACKED4 blocks: x2 (x4 is 0.6 % slower)
#ifndef KS_GEN_UNROLL_PACKED
#define KS_GEN_UNROLL_PACKED 2
#endif

#ifndef KS_VECTOR_KEYS
#define KS_VECTOR_KEYS 0     // Philox round keys in per-thread registers (1) or uniform registers (0)
#endif
#ifndef KS_P0_WIDE
#define KS_P0_WIDE 0         // round-0 product advanced by one IMAD.WIDE accumulate (1) or by a 64-bit add (0)
#endif

namespace ks {

constexpr int kGenUnroll = KS_GEN_UNROLL;
constexpr int kGenUnrollPacked = KS_GEN_UNROLL_PACKED;
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
  int32_t noise_n4;                               // 4*noise_n
  unsigned long long q_addend;                    // 2^32: the "+1" of q = 1 + mulhi(w, qmax), as an IMAD addend
  int32_t maker_spread_max, maker_qty;
  int32_t mom_n, mom_qmax;                        // mom_n = mom_delta+1
  int32_t dmax;                                   // largest |tick - last| any rule can produce
  int32_t fresh;                                  // books are known to be all zero: skip the load
  int32_t force_generic;                          // ablation/test: always use the chunked scan
  int32_t log2C;                                  // cluster kernel only: CTAs per market = 1 << log2C
  int2* trace;                                    // DEVICE [M][S] (price after the step, Vmax), or NULL
  // model 4 (the paper's agent model, A24): class sizes and the marketable threshold;
  // the half spread is maker_spread_max and the makers' qmax is maker_qty
  int32_t paper_n_noise, paper_n_mom, paper_pmkt_q16;
  long long S;                                    // steps to run
  long long orders_per_step;                      // A + number of makers
  // deferred checks (ks_api.cu): the depth bound of a ks_write_books whose result the host has not
  // seen yet (DEVICE word, or NULL), the largest resting depth this run tolerates, and the sticky
  // error flags in MAPPED HOST memory (written on an overflow only)
  const unsigned long long* depth_word;
  unsigned long long depth_limit;
  unsigned long long* host_flags;
  uint32_t rel_stride, rel_side;                  // ks_decoupled_kernel: bytes of ONE relative histogram buffer
                                                  // (sell bins then buy bins) and of one side of it
  uint32_t rel_mk_off, rel_mom_off, rel_mom_side; // ... MIX3: byte offsets, inside a buffer, of the maker bins (one per
                                                  // spread) and of the momentum bins (all quantities per offset, then,
                                                  // rel_mom_side bytes on, the quantities of the agents whose coin says buy)
};

// sticky error flags raised by the kernels (host_flags)
enum : unsigned long long { kFlagStatOverflow = 1ull, kFlagDepthOverflow = 2ull, kFlagNegativeDepth = 4ull };

// u32 x u32 -> u64 as ONE mul.wide.u32 (IMAD.WIDE.U32).  Written as PTX because the compiler,
// given (uint64_t)a * b with a loop-invariant b, hoists the zero-extension of b and then emits a
// 64 x 64 multiply whose (zero) cross term costs an extra add per product.
__device__ __forceinline__ uint64_t mul_wide_u32(uint32_t a, uint32_t b) {
  uint64_t r;
  asm("mul.wide.u32 %0, %1, %2;" : "=l"(r) : "r"(a), "r"(b));
  return r;
}
__device__ __forceinline__ uint32_t hi32(uint64_t x) { return (uint32_t)(x >> 32); }
__device__ __forceinline__ uint32_t lo32(uint64_t x) { return (uint32_t)x; }

// ---------------------------------------------------------------------------------------------
// a1: Philox4x32-10 on ctr = (agent a, step t, market m, 0), with everything that does not
// depend on all three of (a, t, m) hoisted out of the per-event work.
//   round 0:  n0 = hi(M1*m) ^ t ^ k0[0]        (m, t)      n1 = lo(M1*m)              (m)
//             n2 = hi(M0*a) ^ k1[0]            (a)         n3 = lo(M0*a)              (a)
//   round 1:  c0 = hi(M1*n2) ^ n1 ^ k0[1]      (a, m)      c1 = lo(M1*n2)             (a)
//             c2 = hi(M0*n0) ^ n3 ^ k1[1]      (a, m, t)   c3 = lo(M0*n0)             (m, t)
// M1*m is computed once per CTA, M0*n0 once per thread and step.  A thread visits agents
// a, a + a_step, a + 2*a_step, ... so the 64-bit product M0*a is carried as a running sum
// (p0 += M0*a_step: two ALU adds with carry instead of a multiply -- exact, the product of two
// 32-bit numbers never overflows 64 bits).  The 32x32->64 multiplies are what bounds the kernel
// (IMAD.WIDE/IMAD.HI hold an SMSP's fmaheavy pipe for 4 cycles per warp), so per
// event the path issues 16 IMAD.WIDE + 1 IMAD.HI for rounds 1..9 and 2 IMAD.HI for the agent rule.
// ---------------------------------------------------------------------------------------------
// The round keys as the hot loop reads them.  The kernel is bound by the DISPATCH of 16-lane math
// instructions (every IMAD.* / LOP3 / IADD3 holds the shared alu+fma dispatch port for 2 cycles;
// DESIGN.md 7.2), and a LOP3 with a uniform-register operand measures ~0.2 cycles slower than
// one with three vector operands, so the keys are copied once into per-thread registers through
// an opaque move (the compiler would otherwise keep them uniform).
struct Keys { uint32_t k0[10], k1[10]; };

__device__ __forceinline__ Keys load_keys(const KernelParams& P) {
  Keys K;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
#if KS_VECTOR_KEYS
    asm volatile("mov.u32 %0, %1;" : "=r"(K.k0[r]) : "r"(P.k0[r]));
    asm volatile("mov.u32 %0, %1;" : "=r"(K.k1[r]) : "r"(P.k1[r]));
#else
    K.k0[r] = P.k0[r]; K.k1[r] = P.k1[r];
#endif
  }
  return K;
}

struct MarketUniform {   // depends on the market only (plus the launch's keys, carried along)
  uint32_t hm;     // hi(M1*m)
  uint32_t n1k;    // lo(M1*m) ^ k0[1]
  Keys K;          // round keys for the per-event rounds
};
struct StepUniform {     // depends on (market, step)
  uint32_t d2x;    // hi(M0*n0) ^ k1[1]
  uint32_t d3;     // lo(M0*n0)
  uint32_t d3k;    // d3 ^ k1[2]: round 2 xors two uniform words into hi(M0*c0); pre-xored here
};

__device__ __forceinline__ MarketUniform market_uniform(const KernelParams& P, uint32_t market) {
  uint64_t pm = (uint64_t)kPhiloxM1 * market;
  MarketUniform mu;
  mu.hm = hi32(pm);
  mu.n1k = lo32(pm) ^ P.k0[1];
  mu.K = load_keys(P);
  return mu;
}

__device__ __forceinline__ StepUniform step_uniform(const KernelParams& P, const MarketUniform& mu, uint32_t t) {
  uint32_t n0 = mu.hm ^ t ^ P.k0[0];
  uint64_t q0 = (uint64_t)kPhiloxM0 * n0;
  StepUniform u;
  u.d2x = hi32(q0) ^ P.k1[1];
  u.d3 = lo32(q0);
  u.d3k = u.d3 ^ P.k1[2];
  return u;
}

// Philox4x32-10 of agent a from p0 = M0*a (round 0's product).  Outputs w0, w1, w2 (w3 is
// reserved and never computed).  NEED02 = false skips the last round's M0 product and w0 (the
// maker rule reads w1 only).
// rounds 0..8 from p0 = M0*c0_in: the state (c0, c1, c2, c3) that enters the last round
__device__ __forceinline__ void philox_rounds_0_8(const KernelParams& P, const MarketUniform& mu, const StepUniform& u,
                                                  uint64_t p0, uint32_t& c0, uint32_t& c1, uint32_t& c2, uint32_t& c3) {
  {                                       // rounds 0-1
    const uint32_t n2 = hi32(p0) ^ mu.K.k1[0];
    const uint64_t p1 = (uint64_t)kPhiloxM1 * n2;
    c0 = hi32(p1) ^ mu.n1k;
    c1 = lo32(p1);
    c2 = u.d2x ^ lo32(p0);
  }
  {                                       // round 2: c3 = d3 is uniform, d3 ^ k1[2] was pre-xored
    uint64_t a0 = (uint64_t)kPhiloxM0 * c0;
    uint64_t a1 = (uint64_t)kPhiloxM1 * c2;
    uint32_t t0 = hi32(a1) ^ c1 ^ mu.K.k0[2];
    uint32_t t2 = hi32(a0) ^ u.d3k;
    c1 = lo32(a1); c3 = lo32(a0); c0 = t0; c2 = t2;
  }
#pragma unroll
  for (int r = 3; r < 9; ++r) {
    uint64_t a0 = (uint64_t)kPhiloxM0 * c0;
    uint64_t a1 = (uint64_t)kPhiloxM1 * c2;
    uint32_t t0 = hi32(a1) ^ c1 ^ mu.K.k0[r];
    uint32_t t2 = hi32(a0) ^ c3 ^ mu.K.k1[r];
    c1 = lo32(a1);
    c3 = lo32(a0);
    c0 = t0;
    c2 = t2;
  }
}

template <bool NEED02>
__device__ __forceinline__ void philox_from_p0(const KernelParams& P, const MarketUniform& mu, const StepUniform& u,
                                               uint64_t p0, uint32_t& w0, uint32_t& w1, uint32_t& w2) {
  uint32_t c0, c1, c2, c3;
  philox_rounds_0_8(P, mu, u, p0, c0, c1, c2, c3);
  uint64_t a1 = (uint64_t)kPhiloxM1 * c2;
  w1 = lo32(a1);
  if (NEED02) {
    w0 = hi32(a1) ^ c1 ^ mu.K.k0[9];
    w2 = __umulhi(kPhiloxM0, c0) ^ c3 ^ mu.K.k1[9];
  } else {
    w0 = 0; w2 = 0;
  }
}

// PACKED4 contract (A22): all four words of the block of agents 4b..4b+3, p0 = M0*b.
__device__ __forceinline__ void philox_block_from_p0(const KernelParams& P, const MarketUniform& mu,
                                                     const StepUniform& u, uint64_t p0, uint32_t (&w)[4]) {
  uint32_t c0, c1, c2, c3;
  philox_rounds_0_8(P, mu, u, p0, c0, c1, c2, c3);
  const uint64_t a0 = (uint64_t)kPhiloxM0 * c0;
  const uint64_t a1 = (uint64_t)kPhiloxM1 * c2;
  w[0] = hi32(a1) ^ c1 ^ mu.K.k0[9];
  w[1] = lo32(a1);
  w[2] = hi32(a0) ^ c3 ^ mu.K.k1[9];
  w[3] = lo32(a0);
}

// Per-step trace: lane 0 of the clearing warp stages (price, Vmax) of step s in
// shared memory; every 32 steps (and after the last one) the warp flushes the staged entries with
// one coalesced 256-byte store.  gtrace points at this market's S entries.
__device__ __forceinline__ void trace_step(int2* s_trace, int2* gtrace, long long s, long long S, int lane,
                                           int price, int vmax) {
  const int slot = (int)(s & 31);
  if (lane == 0) s_trace[slot] = make_int2(price, vmax);
  __syncwarp();
  if (slot == 31 || s == S - 1) {
    if (lane <= slot) gtrace[s - slot + lane] = s_trace[lane];
    __syncwarp();
  }
}

// a2: add one order to the shared-memory book at byte offset `off` from the start of the [2][L]
// book.  ATOM 0: plain shared-memory reduction (ATOMS.ADD, result unused).  ATOM 1: warp-aggregated
// -- lanes with the same address elect a leader that adds the group's sum (north_star (3)); kept
// as an ablation switch.  ATOM 2: microbenchmark only, no memory access.  ATOM 3: the book is
// split across the CTAs of a cluster (ks_cluster.cuh): remote shared-memory reduction over DSMEM.
struct BookRef {
  int32_t* ptr;        // generic pointer to the book
  uint32_t saddr;      // its 32-bit shared-window address
  int log2L, log2Lc;   // ATOM 3 only: L = 1 << log2L ticks, 1 << log2Lc of them per CTA
#ifdef KS_DEBUG_CHECKS
  uint32_t dbg_lo, dbg_hi;   // shared-window byte range an order may be added to (book, or relative histogram)
  int* dbg_count;            // shared counter of the orders added in the current step
#endif
};

// KS_DEBUG_CHECKS (python -m paper_2606_21784_b200.build --debug-checks -> libkineticsim_dbg.so):
// the library's own bounds and phase checks, in place of compute-sanitizer (closed on this pool,
// profiles/r2_sanitizer.md).  Every order's shared-memory address must lie inside the book (or the
// relative histogram being filled); every book access of the clearing code inside [0, L); and --
// the phase structure of Alg.1 -- when the clearing warp starts on a
// step, EXACTLY the step's orders have been added since it last looked (a missed or early barrier
// shows up as a wrong count).  A failed check prints its location and traps.
#ifdef KS_DEBUG_CHECKS
#define KS_CHECK(cond, what)                                                                                   \
  do {                                                                                                         \
    if (!(cond)) {                                                                                             \
      printf("KS_DEBUG_CHECKS failed: %s (%s:%d) block %d thread %d\n", what, __FILE__, __LINE__, (int)blockIdx.x, \
             (int)threadIdx.x);                                                                                \
      __trap();                                                                                                \
    }                                                                                                          \
  } while (0)
#else
#define KS_CHECK(cond, what) do { } while (0)
#endif

template <int ATOM>
__device__ __forceinline__ void book_add_at(const BookRef& book, uint32_t saddr, int q, int& sink) {
#ifdef KS_DEBUG_CHECKS
  if (ATOM != 2) {
    KS_CHECK(saddr >= book.dbg_lo && saddr + 4u <= book.dbg_hi && (saddr & 3u) == 0u, "order address outside its target array");
    KS_CHECK(q > 0, "order quantity not positive");
    atomicAdd(book.dbg_count, 1);
  }
#endif
  if (ATOM == 0) {
    asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(saddr), "r"(q) : "memory");
  } else if (ATOM == 2) {
    sink ^= (int)saddr * 131 + q;        // no memory access (ks_bench_generate_only)
  } else {
    unsigned act = __activemask();
    unsigned peers = __match_any_sync(act, saddr);
    int sum = __reduce_add_sync(peers, q);
    if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) atomicAdd(book.ptr + ((saddr - book.saddr) >> 2), sum);
  }
}

template <int ATOM>
__device__ __forceinline__ void book_add(const BookRef& book, uint32_t off, int q, int& sink) {
  if (ATOM == 3) {
    const uint32_t word = off >> 2, side = word >> book.log2L, tick = word & ((1u << book.log2L) - 1u);
    const uint32_t rank = tick >> book.log2Lc;
    const uint32_t loc = (side << book.log2Lc) + (tick & ((1u << book.log2Lc) - 1u));
    uint32_t caddr;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(caddr) : "r"(book.saddr + 4u * loc), "r"(rank));
    asm volatile("red.shared::cluster.add.s32 [%0], %1;" ::"r"(caddr), "r"(q) : "memory");
  } else {
    book_add_at<ATOM>(book, book.saddr + off, q, sink);
  }
}

__device__ __forceinline__ int clamp_tick(int x, int L) { return min(max(x, 0), L - 1); }

// Per-step values of the rules that are uniform over the CTA.  bid_lo / ask_lo are absolute
// shared addresses, published once per step by the clearing warp (ks_kernel.cuh, s_ctl) so that
// no thread recomputes them per order.
struct RuleCtx {
  int last, dp, L;
  bool noclamp;          // last - noise_delta >= 0 and last + noise_delta <= L-1: the noise clamp is the identity
  uint32_t bid_lo;       // shared address of bid[last - noise_delta]
  uint32_t ask_lo;       // shared address of ask[last - noise_delta]
  uint32_t bid_last, ask_last;   // shared addresses of bid[last], ask[last] (MIX3 no-clamp paths)
  int mid2;              // model 4: doubled mid price of the resting book (Eq.3); dp = sgn(mid2 - previous mid2)
  int* mkt_flags;        // model 4: shared int[2], set when a marketable buy [0] / sell [1] was generated
  uint32_t rel_s, rel_b; // ATOM 4 / 5: shared addresses of sell bin 0 and of buy bin n-1 of the relative order
                         // histogram being filled (plus 4*lane for the lane-columned layout)
};

// ATOM 4 / 5 (ks_decoupled_kernel): a noise order goes into a PRICE-INDEPENDENT relative histogram
// instead of the book: with o = the offset draw in [0, n), a sell adds to sell[o] and a buy to
// buy[n-1-o], so that for BOTH sides bin i means tick (last - delta) + i (sell tick = last - delta
// + o; buy tick = last + delta - o = last - delta + (n-1-o)).  Only the clearing warp turns bins
// into ticks, when it merges the histogram into the book at the step's price (clamping to the
// grid there).  Integer adds commute, so the combined book is the one the direct path builds.
// ATOM 4: one int32 per bin (byte stride 4); ATOM 5: 32 lane columns per bin (byte stride 128,
// column = lane = bank): the 32 atomics of a warp instruction never share a bank (SURVEY.md S7
// "lane-columned relative histogram").  Same three instructions as the direct no-clamp path.
template <int ATOM>
__device__ __forceinline__ uint32_t rel_bin_addr(const RuleCtx& rc, uint32_t side_word, uint32_t o) {
  constexpr int sh = ATOM == 4 ? 2 : 7;
  return (int32_t)side_word < 0 ? rc.rel_b - (o << sh) : rc.rel_s + (o << sh);
}

// a1 noise rule.  o = mulhi(w1, n), n = 2*delta+1; sell tick = (last - delta) + o, buy tick =
// last - (o - delta) = (last + delta) - o.  q = 1 + mulhi(w2, qmax) is the high word of
// w2*qmax + 2^32: one IMAD.HI with the +1 folded into its 64-bit addend.
// No-clamp path: addr = buy ? &bid[last+delta] - 4*o : &ask[last-delta] + 4*o, which compiles to
// ISETP + IMAD(o, -4, bid_hi) + @P IMAD(o, 4, ask_lo).  The kernel is bound by the number of math
// instructions it dispatches (~1 % of run time per instruction per event), so the
// rule is written for the fewest instructions, whichever pipe runs them (mask-and-xor forms of
// the same address need four or five).
template <int ATOM, bool CLAMP>
__device__ __forceinline__ void noise_order(const KernelParams& P, const BookRef& book, const RuleCtx& rc,
                                            uint32_t w0, uint32_t w1, uint32_t w2, int& sink) {
  const int q = (int)hi32((uint64_t)w2 * (uint32_t)P.noise_qmax + P.q_addend);
  if (ATOM == 4 || ATOM == 5) {
    book_add_at<0>(book, rel_bin_addr<ATOM>(rc, w0, __umulhi(w1, (uint32_t)P.noise_n)), q, sink);
  } else if (!CLAMP) {
    // three instructions: one compare and two multiply-adds of which one is predicated off
    const uint32_t o = __umulhi(w1, (uint32_t)P.noise_n);
    const uint32_t bid_hi = rc.bid_lo + (uint32_t)P.noise_n4 - 4u;            // &bid[last + delta]
    const uint32_t addr = (int32_t)w0 < 0 ? bid_hi - (o << 2) : rc.ask_lo + (o << 2);
    book_add_at<ATOM>(book, addr, q, sink);
  } else {
    const bool buy = (int32_t)w0 < 0;
    const int o = (int)__umulhi(w1, (uint32_t)P.noise_n);
    const int tick = clamp_tick(buy ? (rc.last + P.noise_delta) - o : (rc.last - P.noise_delta) + o, rc.L);
    book_add<ATOM>(book, 4u * (uint32_t)(buy ? tick : tick + rc.L), q, sink);
  }
}

// a1 maker rule: both sides, fixed quantity; only w1 is used.  No-clamp path: s0 = mulhi(w1, smax),
// bid at &bid[last-1] - 4*s0, ask at &ask[last+1] + 4*s0 -- three math instructions.
template <int ATOM, bool CLAMP>
__device__ __forceinline__ void maker_order(const KernelParams& P, const BookRef& book, const RuleCtx& rc,
                                            uint32_t w1, int& sink) {
  const uint32_t s0 = __umulhi(w1, (uint32_t)P.maker_spread_max);
  if (!CLAMP) {
    book_add_at<ATOM>(book, rc.bid_last - 4u - (s0 << 2), P.maker_qty, sink);
    book_add_at<ATOM>(book, rc.ask_last + 4u + (s0 << 2), P.maker_qty, sink);
  } else {
    const int s = 1 + (int)s0;
    book_add<ATOM>(book, 4u * (uint32_t)clamp_tick(rc.last - s, rc.L), P.maker_qty, sink);
    book_add<ATOM>(book, 4u * (uint32_t)(clamp_tick(rc.last + s, rc.L) + rc.L), P.maker_qty, sink);
  }
}

// a1 momentum rule: dp = last - prev is uniform over the market-step.  No-clamp path when the side
// is the same for the whole step (dp != 0): addr = &bid[last] + 4*o or &ask[last] - 4*o.
template <int ATOM, bool CLAMP>
__device__ __forceinline__ void momentum_order(const KernelParams& P, const BookRef& book, const RuleCtx& rc,
                                               uint32_t w0, uint32_t w1, uint32_t w2, int& sink) {
  const uint32_t o = __umulhi(w1, (uint32_t)P.mom_n);
  const int q = (int)hi32((uint64_t)w2 * (uint32_t)P.mom_qmax + P.q_addend);
  if (!CLAMP && rc.dp != 0) {
    book_add_at<ATOM>(book, rc.dp > 0 ? rc.bid_last + (o << 2) : rc.ask_last - (o << 2), q, sink);
  } else {
    const bool buy = rc.dp > 0 ? true : (rc.dp < 0 ? false : ((int32_t)w0 < 0));
    const int tick = clamp_tick(buy ? rc.last + (int)o : rc.last - (int)o, rc.L);
    book_add<ATOM>(book, 4u * (uint32_t)(buy ? tick : tick + rc.L), q, sink);
  }
}

// ---- PACKED4 rules (A22): every draw of an agent out of ONE word by successive
// multiply-extract: o = hi(w*n), x1 = lo(w*n); q-1 = hi(x1*qmax), x2 = lo(x1*qmax); coin = x2>>31.
// Two IMAD.WIDE per agent.  (ptxas splits a mad.wide.u32 with a 64-bit addend into multiply + two
// adds when the multiplier is a uniform register, so the +1 of q is a plain add.)
// No-clamp noise path: m = coin mask (all-ones for a buy); sell tick = (last-delta) + o, buy tick
// = (last-delta) + (n-1-o) = (last-delta+n) + ~o, so addr = base(m) + 4*(o ^ m) with base =
// &ask[last-delta] or &bid[last-delta+n]: SHF + 2 LOP3 + one shift-add.  (The compare-and-
// predicate form that wins in the literal rule measures 8 % SLOWER here: the predicate comes
// out of the second multiply, at the end of the dependency chain.)
template <int ATOM, bool CLAMP>
__device__ __forceinline__ void noise_order_packed(const KernelParams& P, const BookRef& book, const RuleCtx& rc,
                                                   uint32_t w, int& sink) {
  const uint64_t p1 = mul_wide_u32(w, (uint32_t)P.noise_n);
  const uint64_t p2 = mul_wide_u32(lo32(p1), (uint32_t)P.noise_qmax);
  const int q = (int)hi32(p2) + 1;
  const uint32_t o = hi32(p1);
  if (ATOM == 4 || ATOM == 5) {
    book_add_at<0>(book, rel_bin_addr<ATOM>(rc, lo32(p2), o), q, sink);
  } else if (!CLAMP) {
    const uint32_t m = (uint32_t)((int32_t)lo32(p2) >> 31);
    const uint32_t bid_top = rc.bid_lo + (uint32_t)P.noise_n4;
    const uint32_t base = rc.ask_lo ^ (m & (rc.ask_lo ^ bid_top));
    book_add_at<ATOM>(book, base + ((o ^ m) << 2), q, sink);
  } else {
    const bool buy = (int32_t)lo32(p2) < 0;
    const int tick = clamp_tick(buy ? (rc.last + P.noise_delta) - (int)o : (rc.last - P.noise_delta) + (int)o, rc.L);
    book_add<ATOM>(book, 4u * (uint32_t)(buy ? tick : tick + rc.L), q, sink);
  }
}

template <int ATOM>
__device__ __forceinline__ void momentum_order_packed(const KernelParams& P, const BookRef& book, const RuleCtx& rc,
                                                      uint32_t w, int& sink) {
  const uint64_t p1 = mul_wide_u32(w, (uint32_t)P.mom_n);
  const uint64_t p2 = mul_wide_u32(lo32(p1), (uint32_t)P.mom_qmax);
  const int q = (int)hi32(p2) + 1;
  const int o = (int)hi32(p1);
  const bool buy = rc.dp > 0 ? true : (rc.dp < 0 ? false : ((int32_t)lo32(p2) < 0));
  const int tick = clamp_tick(buy ? rc.last + o : rc.last - o, rc.L);
  book_add<ATOM>(book, 4u * (uint32_t)(buy ? tick : tick + rc.L), q, sink);
}

// One agent of type KIND under PACKED4 from its word.
template <int ATOM, int KIND, bool CLAMP>
__device__ __forceinline__ void packed_agent(const KernelParams& P, const BookRef& book, const RuleCtx& rc,
                                             uint32_t w, int& sink) {
  if (KIND == 0)      noise_order_packed<ATOM, CLAMP>(P, book, rc, w, sink);
  else if (KIND == 1) maker_order<ATOM, true>(P, book, rc, w, sink);
  else                momentum_order_packed<ATOM>(P, book, rc, w, sink);
}

// ---- model 4, the paper's agent model (SIII-C; A24), doubled-integer
// prices: round(m2 / 2) half up = (m2 + 1) >> 1 (arithmetic shift = floor).  KIND 0 noise,
// 1 momentum, 2 maker.  `parity` = (a + t) & 1 of this thread's agents (T is even, so it is the
// same for all of them).  Marketable orders go to the grid boundary and raise a flag so that the
// clearing warp widens its window to that boundary.
template <int ATOM, int KIND, bool CLAMP>
__device__ __forceinline__ void paper_order(const KernelParams& P, const BookRef& book, const RuleCtx& rc,
                                            const uint32_t (&w)[4], uint32_t parity, uint32_t& mkt_seen, int& sink) {
  const uint32_t qmax = KIND == 0 ? (uint32_t)P.noise_qmax : (KIND == 1 ? (uint32_t)P.mom_qmax : (uint32_t)P.maker_qty);
  const int q = (int)hi32((uint64_t)w[2] * qmax + P.q_addend);
  const bool buy = KIND == 0 ? (int32_t)w[0] < 0
                 : KIND == 1 ? (rc.dp > 0 ? true : (rc.dp < 0 ? false : ((int32_t)w[0] < 0)))
                             : parity == 0u;
  const bool mkt = KIND != 2 && (int)(w[3] >> 16) < P.paper_pmkt_q16;
  if (!CLAMP) {
    // round(mid + k) = midr + k for an integer k, midr = (mid2 + 1) >> 1 (2k is even), and no
    // price can leave the grid: rc.bid_lo / rc.ask_lo are &bid / &ask[midr - delta], rc.bid_last /
    // rc.ask_last are &bid / &ask[midr]
    uint32_t addr;
    if (KIND == 0) {
      const uint32_t o4 = __umulhi(w[1], (uint32_t)P.noise_n) << 2;
      addr = buy ? rc.bid_lo + o4 : rc.ask_lo + o4;
    } else if (KIND == 1) {
      addr = buy ? rc.bid_last + 4u : rc.ask_last - 4u;
    } else {
      addr = buy ? rc.bid_last - 4u * (uint32_t)P.maker_spread_max : rc.ask_last + 4u * (uint32_t)P.maker_spread_max;
    }
    if (KIND != 2) {
      // branch-free (a divergent branch per event kept ptxas from interleaving the four unrolled
      // events): the edge address by two selects; whether the thread generated ANY marketable order
      // this step is the running minimum of the 16-bit draw, one instruction per event
      // (generate_step_paper compares it once and raises both flags: the clearing warp then reads the
      // depth at both edge ticks, and an edge nobody hit holds none)
      const uint32_t edge = buy ? book.saddr + 4u * (uint32_t)(rc.L - 1) : book.saddr + 4u * (uint32_t)rc.L;   // bid[L-1] / ask[0]
      addr = mkt ? edge : addr;
      mkt_seen = min(mkt_seen, w[3] >> 16);
    }
    book_add_at<ATOM>(book, addr, q, sink);
  } else {
    int p2;
    if (KIND == 0)      p2 = rc.mid2 + 2 * ((int)__umulhi(w[1], (uint32_t)P.noise_n) - P.noise_delta);
    else if (KIND == 1) p2 = rc.mid2 + (buy ? 2 : -2);
    else                p2 = rc.mid2 + (buy ? -2 : 2) * P.maker_spread_max;
    int tick = clamp_tick((p2 + 1) >> 1, rc.L);
    if (KIND != 2) {
      tick = mkt ? (buy ? rc.L - 1 : 0) : tick;
      mkt_seen = min(mkt_seen, w[3] >> 16);
    }
    book_add<ATOM>(book, 4u * (uint32_t)(buy ? tick : tick + rc.L), q, sink);
  }
}

// The agents of one class that a thread visits: first, first + a_step, ... < a_end.  p0 = M0*first;
// n_uniform trips are made by every thread of the CTA (a uniform loop, no per-agent bound
// check), `extra` marks the threads that own one agent more (ragged tail).
struct ClassPlan {
  uint64_t p0;
  uint32_t n_uniform;
  bool extra;
};

__device__ __forceinline__ ClassPlan class_plan(uint32_t first, uint32_t first_of_last_thread, uint32_t a_end,
                                                uint32_t a_step) {
  auto trips = [&](uint32_t f) { return f < a_end ? (a_end - f + a_step - 1u) / a_step : 0u; };
  ClassPlan pl;
  pl.p0 = (uint64_t)kPhiloxM0 * first;
  pl.n_uniform = trips(first_of_last_thread);
  pl.extra = trips(first) > pl.n_uniform;
  return pl;
}

// p + inc as an explicit carry chain, so that it stays one IADD3 + one IADD3.X on the alu pipe and
// is neither turned back into a multiply nor duplicated per unrolled copy.
struct P0Step { uint64_t inc; uint32_t a_step; };   // inc = M0 * a_step

// Advance the round-0 product p0 = M0*a by a_step agents.  KS_P0_WIDE: one IMAD.WIDE with p0 as its
// 64-bit addend -- ONE dispatch slot; the alternative (IADD3 + carry add) spares the fma pipe but
// costs two slots, and dispatch is what binds.
__device__ __forceinline__ uint64_t advance_p0(uint64_t p, uint64_t inc, uint32_t a_step);

__device__ __forceinline__ uint64_t add64_alu(uint64_t p, uint64_t inc) {
  uint32_t lo, hi;
  asm volatile("add.cc.u32 %0, %2, %4;\n\taddc.u32 %1, %3, %5;"
               : "=r"(lo), "=r"(hi)
               : "r"(lo32(p)), "r"(hi32(p)), "r"(lo32(inc)), "r"(hi32(inc)));
  return ((uint64_t)hi << 32) | lo;
}

__device__ __forceinline__ uint64_t advance_p0(uint64_t p, uint64_t inc, uint32_t a_step) {
#if KS_P0_WIDE
  uint64_t r;
  asm volatile("mad.wide.u32 %0, %1, %2, %3;" : "=l"(r) : "r"(a_step), "r"(kPhiloxM0), "l"(p));
  return r;
#else
  return add64_alu(p, inc);
#endif
}

// One agent class of one market-step, rule KIND (0 noise, 1 maker, 2 momentum).
template <int ATOM, int KIND, bool CLAMP>
__device__ __forceinline__ void generate_class(const KernelParams& P, const BookRef& book, const MarketUniform& mu,
                                               const StepUniform& u, const RuleCtx& rc, const ClassPlan& pl,
                                               const P0Step& p0_inc, int& sink) {
  auto one = [&](uint64_t p0) {
    uint32_t w0, w1, w2;
    philox_from_p0<KIND != 1>(P, mu, u, p0, w0, w1, w2);
    if (KIND == 0)      noise_order<ATOM, CLAMP>(P, book, rc, w0, w1, w2, sink);
    else if (KIND == 1) maker_order<ATOM, CLAMP>(P, book, rc, w1, sink);
    else                momentum_order<ATOM, CLAMP>(P, book, rc, w0, w1, w2, sink);
  };
  uint64_t p0 = pl.p0;
#pragma unroll kGenUnroll
  for (uint32_t k = 0; k < pl.n_uniform; ++k) { one(p0); p0 = advance_p0(p0, p0_inc.inc, p0_inc.a_step); }
  if (pl.extra) one(p0);
}

// The same for threads that own at most N <= 4 agents of the class, written for LATENCY (the
// decoupled kernel on an underfilled GPU, where a generating thread holds 1-3 agents and the loop
// above would run its dependent Philox chains one after the other): the N chains are computed
// side by side, unconditionally, and only the atomic is predicated on the agent existing.
template <int ATOM, int N>
__device__ __forceinline__ void generate_class_rel_few(const KernelParams& P, const BookRef& book, const MarketUniform& mu,
                                                       const StepUniform& u, const RuleCtx& rc, const ClassPlan& pl,
                                                       const P0Step& p0_inc, int& sink) {
  const uint32_t n_mine = pl.n_uniform + (pl.extra ? 1u : 0u);
  uint64_t p0 = pl.p0;
  uint32_t addr[N];
  int q[N];
#pragma unroll
  for (uint32_t e = 0; e < N; ++e) {
    uint32_t w0, w1, w2;
    philox_from_p0<true>(P, mu, u, p0, w0, w1, w2);
    q[e] = (int)hi32((uint64_t)w2 * (uint32_t)P.noise_qmax + P.q_addend);
    addr[e] = rel_bin_addr<ATOM>(rc, w0, __umulhi(w1, (uint32_t)P.noise_n));
    p0 = add64_alu(p0, p0_inc.inc);
  }
#pragma unroll
  for (uint32_t e = 0; e < N; ++e)
    if (e < n_mine) book_add_at<0>(book, addr[e], q[e], sink);
}

// G steps of the noise class in one pass over a thread's agents (ks_decoupled_kernel, GROUP): the
// same agent's orders of steps t .. t+G-1, step g into the relative histogram at slot0 + g*stride.
// Written as G plain Philox evaluations on the same p0: everything that does not depend on the
// step -- n2, M1*n2, c0, c1, M0*c0 -- is common to all and is computed once (G = 2: 18 multiplies
// per event instead of 19, G = 4: 17.5; two xors and the 64-bit counter add shared as well).
// Four chains per unrolled trip (4 / G agents).
template <int ATOM, int G>
__device__ __forceinline__ void generate_class_rel_group(const KernelParams& P, const BookRef& book, const MarketUniform& mu,
                                                         const StepUniform (&u)[G], uint32_t slot0, uint32_t stride,
                                                         uint32_t buy_off, const ClassPlan& pl, const P0Step& p0_inc, int& sink) {
  static_assert(ATOM == 4, "plain bins");
  auto one = [&](uint64_t p0) {
    uint32_t w0[G], w1[G], w2[G];
#pragma unroll
    for (int g = 0; g < G; ++g) philox_from_p0<true>(P, mu, u[g], p0, w0[g], w1[g], w2[g]);
#pragma unroll
    for (int g = 0; g < G; ++g) {
      RuleCtx rc;
      rc.rel_s = slot0 + (uint32_t)g * stride;
      rc.rel_b = rc.rel_s + buy_off;
      noise_order<ATOM, false>(P, book, rc, w0[g], w1[g], w2[g], sink);
    }
  };
  uint64_t p0 = pl.p0;
#pragma unroll(4 / G)
  for (uint32_t k = 0; k < pl.n_uniform; ++k) { one(p0); p0 = advance_p0(p0, p0_inc.inc, p0_inc.a_step); }
  if (pl.extra) one(p0);
}

// PACKED4: one class of BLOCKS of four agents.  MIX = false: all noise.  MIX = true: the blocks of
// class CLS are b = 3i + CLS, so agent 4b + j has type (4b + j) mod 3 = (CLS + j) mod 3 -- uniform
// over the warp for every j.
template <int ATOM, bool MIX, int CLS, bool CLAMP>
__device__ __forceinline__ void generate_class_packed(const KernelParams& P, const BookRef& book, const MarketUniform& mu,
                                                      const StepUniform& u, const RuleCtx& rc, const ClassPlan& pl,
                                                      const P0Step& p0_inc, int& sink) {
  auto one = [&](uint64_t p0) {
    uint32_t w[4];
    philox_block_from_p0(P, mu, u, p0, w);
    packed_agent<ATOM, MIX ? (CLS + 0) % 3 : 0, CLAMP>(P, book, rc, w[0], sink);
    packed_agent<ATOM, MIX ? (CLS + 1) % 3 : 0, CLAMP>(P, book, rc, w[1], sink);
    packed_agent<ATOM, MIX ? (CLS + 2) % 3 : 0, CLAMP>(P, book, rc, w[2], sink);
    packed_agent<ATOM, MIX ? (CLS + 3) % 3 : 0, CLAMP>(P, book, rc, w[3], sink);
  };
  uint64_t p0 = pl.p0;
#pragma unroll kGenUnrollPacked
  for (uint32_t k = 0; k < pl.n_uniform; ++k) { one(p0); p0 = advance_p0(p0, p0_inc.inc, p0_inc.a_step); }
  if (pl.extra) one(p0);
}

// PACKED4: the ragged last block (A mod 4 != 0), agents 4b .. A-1, by one thread; types at run time.
template <int ATOM, bool MIX>
__device__ __noinline__ void generate_partial_block_packed(const KernelParams& P, const BookRef& book,
                                                           const MarketUniform& mu, const StepUniform& u,
                                                           const RuleCtx& rc, int& sink) {
  const uint32_t b = (uint32_t)P.A >> 2, rem = (uint32_t)P.A & 3u;
  uint32_t w[4];
  philox_block_from_p0(P, mu, u, (uint64_t)kPhiloxM0 * b, w);
  for (uint32_t j = 0; j < rem; ++j) {
    const uint32_t kind = MIX ? (4u * b + j) % 3u : 0u;
    const uint32_t wj = j == 0 ? w[0] : (j == 1 ? w[1] : w[2]);
    if (kind == 0)      packed_agent<ATOM, 0, true>(P, book, rc, wj, sink);
    else if (kind == 1) packed_agent<ATOM, 1, true>(P, book, rc, wj, sink);
    else                packed_agent<ATOM, 2, true>(P, book, rc, wj, sink);
  }
}

// The per-thread plans of a launch: MODEL 0 one class (a = tid + k*T), MODEL 1 three classes
// (agent a = 3j + c has type c, j = tid + k*T; each class runs in its own warp-uniform loop --
// integer atomics commute, so the agent -> thread mapping cannot change a byte of the result).
template <int MODEL>
struct GenPlan {
  ClassPlan cls[MODEL == 0 ? 1 : 3];
  P0Step p0_inc;         // a_step and M0 * a_step
};

// `count` = number of items the classes enumerate: agents (literal contract) or full blocks of four
// agents (PACKED4).
template <int MODEL>
__device__ __forceinline__ GenPlan<MODEL> gen_plan(uint32_t count, int tid, int T) {
  GenPlan<MODEL> g;
  if (MODEL == 0) {
    g.p0_inc.a_step = (uint32_t)T;
    g.p0_inc.inc = (uint64_t)kPhiloxM0 * (uint32_t)T;
    g.cls[0] = class_plan((uint32_t)tid, (uint32_t)(T - 1), count, (uint32_t)T);
  } else {
    const uint32_t st = 3u * (uint32_t)T;
    g.p0_inc.a_step = st;
    g.p0_inc.inc = (uint64_t)kPhiloxM0 * st;
#pragma unroll
    for (int c = 0; c < (MODEL == 0 ? 1 : 3); ++c)
      g.cls[c] = class_plan(3u * (uint32_t)tid + (uint32_t)c, 3u * (uint32_t)(T - 1) + (uint32_t)c, count, st);
  }
  // hide that p0_inc is a product: otherwise p0 += p0_inc is turned back into IMAD.WIDE(M0, a_step, p0)
  asm volatile("" : "+l"(g.p0_inc.inc));
  return g;
}

// The three-type population (MIX3) for the decoupled kernel, G steps per pass: every rule's order
// is price-independent once it is expressed RELATIVE to the price the step will start from --
//   noise     sell[o] / buy[n-1-o] as above;
//   maker     one spread draw s0: bid at last-1-s0 AND ask at last+1+s0 with the same quantity ->
//             ONE bin mk[s0] (the clearing warp adds it to both sides);
//   momentum  offset o and quantity q; the side is sgn(last - prev), known only when the step is
//             cleared -> all[o] += q, and coin[o] += q for the agents whose coin (w0's top bit)
//             says buy, which decides only when last == prev.
// Same draws, same integer sums as momentum_order / maker_order / noise_order (the clearing warp's
// merge applies the clamp).  Classes as in generate_step<1>: agent 3j + c has type c.
template <int G>
__device__ __forceinline__ void generate_mix3_rel_group(const KernelParams& P, const BookRef& book, const MarketUniform& mu,
                                                        const StepUniform (&u)[G], uint32_t slot0, uint32_t stride,
                                                        uint32_t buy_off, const GenPlan<1>& g3, int& sink) {
  auto noise = [&](uint64_t p0) {
    uint32_t w0[G], w1[G], w2[G];
#pragma unroll
    for (int g = 0; g < G; ++g) philox_from_p0<true>(P, mu, u[g], p0, w0[g], w1[g], w2[g]);
#pragma unroll
    for (int g = 0; g < G; ++g) {
      RuleCtx rc;
      rc.rel_s = slot0 + (uint32_t)g * stride;
      rc.rel_b = rc.rel_s + buy_off;
      noise_order<4, false>(P, book, rc, w0[g], w1[g], w2[g], sink);
    }
  };
  auto maker = [&](uint64_t p0) {
    uint32_t w0, w1[G], w2;
#pragma unroll
    for (int g = 0; g < G; ++g) philox_from_p0<false>(P, mu, u[g], p0, w0, w1[g], w2);
#pragma unroll
    for (int g = 0; g < G; ++g)
      book_add_at<0>(book, slot0 + (uint32_t)g * stride + P.rel_mk_off + (__umulhi(w1[g], (uint32_t)P.maker_spread_max) << 2),
                     P.maker_qty, sink);
  };
  auto momentum = [&](uint64_t p0) {
    uint32_t w0[G], w1[G], w2[G];
#pragma unroll
    for (int g = 0; g < G; ++g) philox_from_p0<true>(P, mu, u[g], p0, w0[g], w1[g], w2[g]);
#pragma unroll
    for (int g = 0; g < G; ++g) {
      const int q = (int)hi32((uint64_t)w2[g] * (uint32_t)P.mom_qmax + P.q_addend);
      const uint32_t a = slot0 + (uint32_t)g * stride + P.rel_mom_off + (__umulhi(w1[g], (uint32_t)P.mom_n) << 2);
      book_add_at<0>(book, a, q, sink);
      if ((int32_t)w0[g] < 0) book_add_at<0>(book, a + P.rel_mom_side, q, sink);
    }
  };
  auto run = [&](const ClassPlan& pl, auto one) {
    uint64_t p0 = pl.p0;
#pragma unroll(4 / G)
    for (uint32_t k = 0; k < pl.n_uniform; ++k) { one(p0); p0 = advance_p0(p0, g3.p0_inc.inc, g3.p0_inc.a_step); }
    if (pl.extra) one(p0);
  };
  run(g3.cls[0], noise);
  run(g3.cls[1], maker);
  run(g3.cls[2], momentum);
}

template <int ATOM, int KIND, bool CLAMP>
__device__ __forceinline__ void generate_class_paper(const KernelParams& P, const BookRef& book, const MarketUniform& mu,
                                                     const StepUniform& u, const RuleCtx& rc, const ClassPlan& pl,
                                                     const P0Step& p0_inc, uint32_t parity, uint32_t& mkt_seen, int& sink) {
  auto one = [&](uint64_t p0) {
    uint32_t w[4];
    philox_block_from_p0(P, mu, u, p0, w);
    paper_order<ATOM, KIND, CLAMP>(P, book, rc, w, parity, mkt_seen, sink);
  };
  uint64_t p0 = pl.p0;
#pragma unroll kGenUnroll
  for (uint32_t k = 0; k < pl.n_uniform; ++k) { one(p0); p0 = advance_p0(p0, p0_inc.inc, p0_inc.a_step); }
  if (pl.extra) one(p0);
}

// model 4: three classes on contiguous agent ranges [0, n_noise), [n_noise, n_noise + n_mom), [.., A)
__device__ __forceinline__ GenPlan<2> gen_plan_paper(const KernelParams& P, int tid, int T) {
  GenPlan<2> g;
  const uint32_t e0 = (uint32_t)P.paper_n_noise, e1 = e0 + (uint32_t)P.paper_n_mom, e2 = (uint32_t)P.A;
  g.p0_inc.a_step = (uint32_t)T;
  g.p0_inc.inc = (uint64_t)kPhiloxM0 * (uint32_t)T;
  g.cls[0] = class_plan((uint32_t)tid, (uint32_t)(T - 1), e0, (uint32_t)T);
  g.cls[1] = class_plan(e0 + (uint32_t)tid, e0 + (uint32_t)(T - 1), e1, (uint32_t)T);
  g.cls[2] = class_plan(e1 + (uint32_t)tid, e1 + (uint32_t)(T - 1), e2, (uint32_t)T);
  asm volatile("" : "+l"(g.p0_inc.inc));
  return g;
}

template <int ATOM>
__device__ __forceinline__ void generate_step_paper(const KernelParams& P, const BookRef& book, const MarketUniform& mu,
                                                    const StepUniform& u, const RuleCtx& rc, const GenPlan<2>& g,
                                                    int tid, uint32_t t, int& sink) {
  const uint32_t maker_first = (uint32_t)P.paper_n_noise + (uint32_t)P.paper_n_mom + (uint32_t)tid;
  const uint32_t par = (maker_first + t) & 1u;
  uint32_t mkt_seen = 0x10000u;                        // smallest 16-bit marketable draw among this thread's noise / momentum agents (none: 2^16)
  if (rc.noclamp) {
    generate_class_paper<ATOM, 0, false>(P, book, mu, u, rc, g.cls[0], g.p0_inc, 0u, mkt_seen, sink);
    generate_class_paper<ATOM, 1, false>(P, book, mu, u, rc, g.cls[1], g.p0_inc, 0u, mkt_seen, sink);
    generate_class_paper<ATOM, 2, false>(P, book, mu, u, rc, g.cls[2], g.p0_inc, par, mkt_seen, sink);
  } else {
    generate_class_paper<ATOM, 0, true>(P, book, mu, u, rc, g.cls[0], g.p0_inc, 0u, mkt_seen, sink);
    generate_class_paper<ATOM, 1, true>(P, book, mu, u, rc, g.cls[1], g.p0_inc, 0u, mkt_seen, sink);
    generate_class_paper<ATOM, 2, true>(P, book, mu, u, rc, g.cls[2], g.p0_inc, par, mkt_seen, sink);
  }
  if ((int)mkt_seen < P.paper_pmkt_q16) { rc.mkt_flags[0] = 1; rc.mkt_flags[1] = 1; }
}

// The highest tick < `from` with bid depth (-1 if none) / the lowest tick >= `from` with ask depth
// (L if none): chunked warp scans, used by model 4 when the cleared window holds no depth on a
// side and the exact best quote (Eq.3) lies outside it.
template <class IO>
static __device__ __noinline__ int best_bid_below(const IO& io, int L, int from, int lane) {
  for (int c = (from - 1) & ~127; from > 0 && c >= 0; c -= 128) {
    const int t = c + 4 * lane;
    int best = -1;
    if (t < L) {
      const int4 v = io.ld4(0, t);
      const int vals[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int j = 0; j < 4; ++j) if (vals[j] > 0 && t + j < from) best = t + j;
    }
    best = __reduce_max_sync(0xffffffffu, best);
    if (best >= 0) return best;
  }
  return -1;
}

template <class IO>
static __device__ __noinline__ int best_ask_from(const IO& io, int L, int from, int lane) {
  for (int c = max(from, 0) & ~127; c < L; c += 128) {
    const int t = c + 4 * lane;
    int best = 0x7fffffff;
    if (t < L) {
      const int4 v = io.ld4(1, t);
      const int vals[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int j = 3; j >= 0; --j) if (vals[j] > 0 && t + j >= from) best = t + j;
    }
    best = __reduce_min_sync(0xffffffffu, best);
    if (best != 0x7fffffff) return best;
  }
  return L;
}

// a1 + a2 for one market-step: every thread of the CTA generates the orders of its agents.
// `first_thread`: this is thread 0 of the market's thread set (owns PACKED4's ragged last block).
template <int MODEL, int ATOM, bool PACKED>
__device__ __forceinline__ void generate_step(const KernelParams& P, const BookRef& book, const MarketUniform& mu,
                                              const StepUniform& u, const RuleCtx& rc, const GenPlan<MODEL>& g,
                                              bool first_thread, int& sink) {
  const bool fast = ATOM != 3 && rc.noclamp;
  if (!PACKED) {
    if (fast) generate_class<ATOM, 0, false>(P, book, mu, u, rc, g.cls[0], g.p0_inc, sink);
    else      generate_class<ATOM, 0, true >(P, book, mu, u, rc, g.cls[0], g.p0_inc, sink);
    if (MODEL == 1) {
      if (fast) {
        generate_class<ATOM, 1, false>(P, book, mu, u, rc, g.cls[MODEL == 0 ? 0 : 1], g.p0_inc, sink);
        generate_class<ATOM, 2, false>(P, book, mu, u, rc, g.cls[MODEL == 0 ? 0 : 2], g.p0_inc, sink);
      } else {
        generate_class<ATOM, 1, true>(P, book, mu, u, rc, g.cls[MODEL == 0 ? 0 : 1], g.p0_inc, sink);
        generate_class<ATOM, 2, true>(P, book, mu, u, rc, g.cls[MODEL == 0 ? 0 : 2], g.p0_inc, sink);
      }
    }
  } else {
    if (MODEL == 0) {
      if (fast) generate_class_packed<ATOM, false, 0, false>(P, book, mu, u, rc, g.cls[0], g.p0_inc, sink);
      else      generate_class_packed<ATOM, false, 0, true >(P, book, mu, u, rc, g.cls[0], g.p0_inc, sink);
    } else {
      if (fast) {
        generate_class_packed<ATOM, true, 0, false>(P, book, mu, u, rc, g.cls[0], g.p0_inc, sink);
        generate_class_packed<ATOM, true, 1, false>(P, book, mu, u, rc, g.cls[MODEL == 0 ? 0 : 1], g.p0_inc, sink);
        generate_class_packed<ATOM, true, 2, false>(P, book, mu, u, rc, g.cls[MODEL == 0 ? 0 : 2], g.p0_inc, sink);
      } else {
        generate_class_packed<ATOM, true, 0, true>(P, book, mu, u, rc, g.cls[0], g.p0_inc, sink);
        generate_class_packed<ATOM, true, 1, true>(P, book, mu, u, rc, g.cls[MODEL == 0 ? 0 : 1], g.p0_inc, sink);
        generate_class_packed<ATOM, true, 2, true>(P, book, mu, u, rc, g.cls[MODEL == 0 ? 0 : 2], g.p0_inc, sink);
      }
    }
    if ((P.A & 3) != 0 && first_thread) generate_partial_block_packed<ATOM, MODEL == 1>(P, book, mu, u, rc, sink);
  }
}

// The rule context of a step from the market state (every thread computes the same values).
__device__ __forceinline__ RuleCtx rule_ctx(const KernelParams& P, const BookRef& book, int last, int prev) {
  RuleCtx rc;
  rc.last = last; rc.dp = last - prev; rc.L = P.L;
  rc.noclamp = (last - P.dmax >= 0) && (last + P.dmax <= P.L - 1);   // no rule can leave the grid
  rc.bid_lo = book.saddr + 4u * (uint32_t)(last - P.noise_delta);
  rc.ask_lo = book.saddr + 4u * (uint32_t)(P.L + last - P.noise_delta);
  rc.bid_last = rc.bid_lo + 4u * (uint32_t)P.noise_delta;
  rc.ask_last = rc.ask_lo + 4u * (uint32_t)P.noise_delta;
  return rc;
}

// Book accessors of the clearing code: 16-byte vectors of 4 consecutive ticks of one side
// (side 0 = bid, 1 = ask), tick a multiple of 4.  LocalBook: the whole [2][L] book in this CTA's
// shared memory.  ClusterBook (ks_cluster.cuh): the book split across the CTAs of a cluster.
struct LocalBook {
  int32_t* book;
  int L;
  __device__ __forceinline__ int4 ld4(int side, int tick) const {
    KS_CHECK(tick >= 0 && tick + 4 <= L && (tick & 3) == 0, "clearing: vector load outside the grid");
    return *reinterpret_cast<const int4*>((side ? book + L : book) + tick);
  }
  __device__ __forceinline__ void st4(int side, int tick, int4 v) const {
    KS_CHECK(tick >= 0 && tick + 4 <= L && (tick & 3) == 0, "clearing: vector store outside the grid");
    KS_CHECK(v.x >= 0 && v.y >= 0 && v.z >= 0 && v.w >= 0, "clearing: negative residual depth");
    *reinterpret_cast<int4*>((side ? book + L : book) + tick) = v;
  }
  __device__ __forceinline__ int ld1(int side, int tick) const {
    KS_CHECK(tick >= 0 && tick < L, "clearing: load outside the grid");
    return (side ? book + L : book)[tick];
  }
  __device__ __forceinline__ void st1(int side, int tick, int v) const {
    KS_CHECK(tick >= 0 && tick < L && v >= 0, "clearing: store outside the grid or negative depth");
    (side ? book + L : book)[tick] = v;
  }
};

// ---------------------------------------------------------------------------------------------
// a3-a5, one warp, window of at most 32*K ticks starting at `base` (a multiple of K).
// Lane i owns ticks base + i*K .. base + i*K + K-1 in registers.
//   D[p] = (bids of higher lanes) + (own bids at ticks >= p)      Eq.1, suffix
//   S[p] = (asks of lower lanes)  + (own asks at ticks <= p)      Eq.1, prefix
//   V = min(D, S); Vmax by REDUX max; p* = lowest tick attaining it
//   residual: bid <- min(bid, max(0, D - Vmax)), ask <- min(ask, max(0, S - Vmax))
// Also returns, per lane, the candidates for the bounds of the residual book inside the window
// (LaneBounds; reduce_bounds turns them into bmax: highest tick with bid depth, else base-1, and
// amin: lowest tick with ask depth, else the end of the window).  The two reductions are kept out
// of these functions so that the caller can publish the new price first (ks_kernel.cuh): nothing
// on the step's critical path needs them.
// ---------------------------------------------------------------------------------------------
struct LaneBounds { int lb, la; };     // highest own tick with bid depth (-1) / lowest with ask depth (INT_MAX)

__device__ __forceinline__ void reduce_bounds(const LaneBounds& c, int base, int wend, int& bmax_new, int& amin_new) {
  bmax_new = __reduce_max_sync(0xffffffffu, c.lb);
  amin_new = __reduce_min_sync(0xffffffffu, c.la);
  if (bmax_new < 0) bmax_new = base - 1;
  if (amin_new == 0x7fffffff) amin_new = wend;
}

// EXT (model 4's marketable orders): depth that rests OUTSIDE the window but counts
// towards every profile value inside it -- ext.b = the marketable buys at tick L-1 (above the
// window's top: part of D[p] for every p), ext.a = the marketable sells at tick 0 (below its base:
// part of S[p] for every p) -- so that one marketable order does not widen the scan to the grid
// edge.  The window's result is the full-grid result of Eq.1-2 iff
//   ext.b <= S[top]                 (else the buys would reach asks resting above the window), and
//   ext.a == 0, or ext.a <= D[base] and Vmax > ext.a   (else they would reach bids below it; and
//                                    with Vmax == ext.a the lowest-tick tie-break picks a tick
//                                    below the window -- tick 0 itself);
// then both are filled completely (Vmax >= V[top] >= ext.b, Vmax > ext.a) and their ticks end empty.
// The functions return false -- having written nothing -- when the condition fails; the caller
// falls back to the scan that reaches the edge.
struct ExtDepth { int b, a; };

// INC: ib[j] / ia[j] are added to the loaded bid / ask depth of the lane's j-th tick before the
// clearing (the decoupled kernel's incoming orders, fused into the scan instead of being merged
// into the book first); the residual is then stored even when nothing traded.
template <int K, class IO, bool INC = false, bool EXT = false>
__device__ __forceinline__ bool clear_window(const IO& io, int L, int base, int lane,
                                             int& vmax, int& pstar, LaneBounds& lbnd,
                                             const int* ib = nullptr, const int* ia = nullptr,
                                             ExtDepth ext = ExtDepth{0, 0}) {
  static_assert(K % 4 == 0, "K must be a multiple of 4 (16-byte shared-memory vectors)");
  const unsigned FULL = 0xffffffffu;
  const int tick0 = base + lane * K;
  const bool in = tick0 < L;            // L and base are multiples of K: a lane is all in or all out
  int b[K], a[K];
#pragma unroll
  for (int v = 0; v < K / 4; ++v) {
    int4 vb = make_int4(0, 0, 0, 0), va = make_int4(0, 0, 0, 0);
    if (in) {
      vb = io.ld4(0, tick0 + 4 * v);
      va = io.ld4(1, tick0 + 4 * v);
    }
    b[4 * v] = vb.x; b[4 * v + 1] = vb.y; b[4 * v + 2] = vb.z; b[4 * v + 3] = vb.w;
    a[4 * v] = va.x; a[4 * v + 1] = va.y; a[4 * v + 2] = va.z; a[4 * v + 3] = va.w;
  }
  if (INC) {
#pragma unroll
    for (int j = 0; j < K; ++j) { b[j] += ib[j]; a[j] += ia[j]; }
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
  const int D0 = sufb + (EXT ? ext.b : 0), S0 = prea - ta + (EXT ? ext.a : 0);
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
  if (EXT) {
    const int Dbase = __shfl_sync(FULL, D0, 0), Stop = __shfl_sync(FULL, S0 + ta, 31);
    if (ext.b > Stop || (ext.a != 0 && (ext.a > Dbase || vmax <= ext.a))) return false;
  }
  int lb = -1, la = 0x7fffffff;
  if (vmax > 0 || INC) {
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
    }
    if (in) {
#pragma unroll
      for (int v = 0; v < K / 4; ++v) {
        io.st4(0, tick0 + 4 * v, make_int4(b[4 * v], b[4 * v + 1], b[4 * v + 2], b[4 * v + 3]));
        io.st4(1, tick0 + 4 * v, make_int4(a[4 * v], a[4 * v + 1], a[4 * v + 2], a[4 * v + 3]));
      }
    }
  }
#pragma unroll
  for (int j = 0; j < K; ++j) {
    if (b[j] > 0) lb = tick0 + j;                      // ascending: the highest wins
    if (a[K - 1 - j] > 0) la = tick0 + K - 1 - j;      // descending: the lowest wins
  }
  lbnd.lb = lb; lbnd.la = la;
  return true;
}

// One step of an inclusive warp scan with the shuffle's own range predicate: x += value of the
// lane d below (scan_up) / d above (scan_down) when that lane exists -- SHFL + one predicated add
// (the CUDA intrinsics hide the predicate and need a compare or a mask besides).
__device__ __forceinline__ int scan_up_add(int x, int d) {
  int r;
  asm volatile("{\n\t.reg .pred p;\n\t.reg .s32 t;\n\tshfl.sync.up.b32 t|p, %1, %2, 0, 0xffffffff;\n\tmov.s32 %0, %1;\n\t@p add.s32 %0, %1, t;\n\t}"
               : "=r"(r) : "r"(x), "r"(d));
  return r;
}
__device__ __forceinline__ int scan_down_add(int x, int d) {
  int r;
  asm volatile("{\n\t.reg .pred p;\n\t.reg .s32 t;\n\tshfl.sync.down.b32 t|p, %1, %2, 31, 0xffffffff;\n\tmov.s32 %0, %1;\n\t@p add.s32 %0, %1, t;\n\t}"
               : "=r"(r) : "r"(x), "r"(d));
  return r;
}

// a3-a5 for a window of at most 32*R ticks starting at `base` (ANY alignment), as R rows of 32
// ticks: lane i owns ticks base + i, base + 32 + i, ... -- one tick per lane and row, so there is
// no per-lane inner loop, every shared-memory access is a conflict-free 32-bit row, and the 2R
// scans (suffix of bids, prefix of asks, per row) are independent chains that the warp overlaps;
// the rows are then chained through their totals.  R = 1 is the short path of C1 / C3 (delta = 8),
// R = 2 covers C2 (delta = 16: 33 ticks).  Same definitions as clear_window.  INC: ib[r] / ia[r]
// are added to the loaded depth of the lane's tick in row r before the clearing (the decoupled
// kernel's incoming orders, fused into the scan).
template <int R, class IO, bool INC = false, bool EXT = false>
__device__ __forceinline__ bool clear_rows(const IO& io, int L, int base, int lane,
                                           int& vmax, int& pstar, LaneBounds& lbnd,
                                           const int* ib = nullptr, const int* ia = nullptr,
                                           ExtDepth ext = ExtDepth{0, 0}) {
  const unsigned FULL = 0xffffffffu;
  int tick[R], b0[R], a0[R], b[R], a[R], D[R], S[R];
  bool in[R];
#pragma unroll
  for (int r = 0; r < R; ++r) {
    tick[r] = base + 32 * r + lane;
    in[r] = tick[r] < L;
    b0[r] = in[r] ? io.ld1(0, tick[r]) : 0;
    a0[r] = in[r] ? io.ld1(1, tick[r]) : 0;
  }
#pragma unroll
  for (int r = 0; r < R; ++r) {
    b[r] = b0[r] + (INC ? ib[r] : 0);
    a[r] = a0[r] + (INC ? ia[r] : 0);
    D[r] = b[r]; S[r] = a[r];
  }
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
#pragma unroll
    for (int r = 0; r < R; ++r) { D[r] = scan_down_add(D[r], d); S[r] = scan_up_add(S[r], d); }
  }
  if (R > 1) {                          // chain the rows: asks of the lower rows, bids of the higher rows
    int rowA[R], rowB[R];
#pragma unroll
    for (int r = 0; r < R; ++r) { rowA[r] = __shfl_sync(FULL, S[r], 31); rowB[r] = __shfl_sync(FULL, D[r], 0); }
    int carryA = 0, carryB = 0;
#pragma unroll
    for (int r = 1; r < R; ++r) { carryA += rowA[r - 1]; S[r] += carryA; }
#pragma unroll
    for (int r = R - 2; r >= 0; --r) { carryB += rowB[r + 1]; D[r] += carryB; }
  }
  if (EXT) {
#pragma unroll
    for (int r = 0; r < R; ++r) { D[r] += ext.b; S[r] += ext.a; }
  }
  int V[R], bestV = 0;
#pragma unroll
  for (int r = 0; r < R; ++r) { V[r] = min(D[r], S[r]); bestV = max(bestV, V[r]); }
  vmax = __reduce_max_sync(FULL, bestV);
  int cand = 0x7fffffff;
#pragma unroll
  for (int r = R - 1; r >= 0; --r) if (V[r] == vmax) cand = tick[r];      // descending: the lowest row wins
  pstar = __reduce_min_sync(FULL, vmax > 0 ? cand : 0x7fffffff);
  if (EXT) {
    const int Dbase = __shfl_sync(FULL, D[0], 0), Stop = __shfl_sync(FULL, S[R - 1], 31);
    if (ext.b > Stop || (ext.a != 0 && (ext.a > Dbase || vmax <= ext.a))) return false;
  }
  if (vmax > 0) {
#pragma unroll
    for (int r = 0; r < R; ++r) { b[r] = min(b[r], max(0, D[r] - vmax)); a[r] = min(a[r], max(0, S[r] - vmax)); }
  }
  int lb = -1, la = 0x7fffffff;
#pragma unroll
  for (int r = 0; r < R; ++r) {
    if (in[r] && b[r] != b0[r]) io.st1(0, tick[r], b[r]);
    if (in[r] && a[r] != a0[r]) io.st1(1, tick[r], a[r]);
    if (b[r] > 0) lb = tick[r];                                            // ascending: the highest wins
    if (a[R - 1 - r] > 0) la = tick[R - 1 - r];                            // descending: the lowest wins
  }
  lbnd.lb = lb; lbnd.la = la;
  return true;
}

// General window of any width: chunks of 128 ticks, three passes (total bid depth; profiles and
// arg max; residual and bounds).  Slow path: first step after a ks_write_books, or a window wider
// than 256 ticks.  Same definitions as clear_window.
template <class IO>
static __device__ __noinline__ void clear_generic(const IO& io, int L, int base, int top, int lane,
                                           int& vmax, int& pstar, LaneBounds& lbnd) {
  const unsigned FULL = 0xffffffffu;
  // pass 0: total bid depth of the window
  int tbsum = 0;
  for (int c = base; c <= top; c += 128) {
    int t = c + lane * 4;
    if (t < L) { int4 vb = io.ld4(0, t); tbsum += vb.x + vb.y + vb.z + vb.w; }
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
      if (in) { vb = io.ld4(0, t); va = io.ld4(1, t); }
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
        io.st4(0, t, make_int4(b[0], b[1], b[2], b[3]));
        io.st4(1, t, make_int4(a[0], a[1], a[2], a[3]));
      }
      carryB += __shfl_sync(FULL, preb, 31);
      carryA += __shfl_sync(FULL, prea, 31);
    }
    if (pass == 1) {
      vmax = __reduce_max_sync(FULL, bestV);
      pstar = __reduce_min_sync(FULL, bestV == vmax ? bestp : 0x7fffffff);
    }
  }
  lbnd.lb = lb; lbnd.la = la;
}

}  // namespace ks
