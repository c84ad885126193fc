/*
 * ks_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU oracle for the hot path of KineticSim
 * (arxiv/paper_2606_21784): persistent, state-carrying uniform-price call-auction
 * clearing for independent limit-order-book markets.  It is the plain definition
 * written out, O(A + L) per market-step with 64-bit sums, and shares NO code,
 * headers, tables or constants with the CUDA path under paper_2606_21784_b200/.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.
 *
 * What follows which passage (PAPER.md line numbers; SURVEY.md = /root/repo/SURVEY.md):
 *   ko_clear_step      Eq.1 cumulative demand/supply, Eq.2
 *                      volume-maximising price, tie -> lowest tick,
 *                      price-priority allocation and residual carry (PAPER.md:343-354,
 *                      PAPER.md:55).
 *   ko_gen_orders      agent rules shaped after SIII-C in the integer
 *                      form BASELINE.json `configs` fixes, driven
 *                      by a counter-based generator (SIII-G) which
 *                      BASELINE.json's north_star replaces by Philox4x32-10 keyed by
 *                      (seed, market, step, agent).
 *   ko_run_markets     Alg.1: per step all agents see the state as it
 *                      was at the start of the step (l.6-7), orders are added to the book
 *                      (l.10-13), the combined book is cleared (l.15-21) and the residual
 *                      becomes the next step's resting book (l.22); reading A2 of
 *                      DESIGN.md (combined = resting + incoming).
 *   ko_derived         fp64 statistics derived from the integer sums (PAPER.md:302,
 *                      PAPER.md:442-456).
 *   ko_run_markets_traced, ko_trace_stats   per-step (price, volume) trace and the return
 *                      statistics of SIV-J (Fig.7): volatility, excess
 *                      kurtosis, volume per step, ACF of r and |r| (reading A23).
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors,
 * the paper's worked example Eq.11-18, brute-force Eq.1-2 on tiny books, greedy
 * best-bid/best-ask matching, closed forms, per-step invariants, a numpy return
 * series for the derived statistics; for the PACKED4 draw contract (models 2, 3) the
 * first four orders by hand from KAT #1 and the exact mixed-radix identity
 * (tests/test_oracle_packed.py); for model 4 (ko_gen_orders_paper) one hand-derived
 * order per class and branch from KAT #1 -- noise, momentum rising / falling / flat,
 * integer and half-tick mids, marketable both ways, maker -- and the momentum rule seen
 * through the run loop on a book whose mid differs from the last price
 * (tests/golden/paper_model_first_order.txt, tests/test_oracle_paper_model.py).
 * Parity unpinned: the paper's own aggregate numbers (Table II, Fig.7) -- its agent
 * parameters and its RNG hash are not given.
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>
#include <stdlib.h>
#include <math.h>

#define KO_API __attribute__((visibility("default")))

/* The oracle's own parameter block (field order is this file's business; the
 * Python wrapper oracle/ks_oracle.py fills it field by field). */
typedef struct {
  int32_t model;            /* 0 = zero-intelligence (all noise), 1 = three types by a mod 3;
                               2, 3 = the same rules under the PACKED4 draw contract (see
                               ko_gen_orders)                                                */
  int32_t noise_delta;      /* noise offset uniform in [-delta, +delta]                      */
  int32_t noise_qmax;       /* noise quantity uniform in 1..qmax                             */
  int32_t maker_spread_max; /* maker spread uniform in 1..spread_max                         */
  int32_t maker_qty;        /* maker fixed quantity on each side                             */
  int32_t mom_delta;        /* momentum offset uniform in [0, delta]                         */
  int32_t mom_qmax;         /* momentum quantity uniform in 1..qmax                          */
  int32_t init_price;       /* < 0 -> L/2                                                    */
  /* model 4 only (the paper's own agent model, ko_gen_orders_paper) */
  int32_t paper_n_mom;      /* number of momentum agents                                     */
  int32_t paper_n_maker;    /* number of market makers                                       */
  int32_t paper_pmkt_q16;   /* P_mkt = paper_pmkt_q16 / 65536                                */
} ko_params;

/* record field indices (SURVEY.md Appendix A "Stats record") */
enum { F_STEPS = 0, F_NTRADES, F_SUMVOL, F_SUMPX, F_SUMPX2, F_SUMPXVOL, F_SUMRET, F_SUMRET2,
       F_SUMRET3, F_SUMRET4, F_SUBBUY, F_SUBSELL, F_LAST, F_PREV, F_HASH, F_NORDERS };

/* ------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2, 3",
 * SC'11), the generator BASELINE.json's north_star (1) mandates in place of the paper's
 * SplitMix64.  One round: (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2,
 * c' = (hi1^c1^k0, lo1, hi0^c3^k1, lo0); the key is bumped by the Weyl constants between
 * rounds.  Ten rounds.
 * ---------------------------------------------------------------------------------------- */
KO_API void ko_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* uniform integer in [0, n) from a 32-bit word: floor(u * n) with u = w / 2^32 exactly
 * ("q = 1 + floor(u * q_max), u ~ U[0,1)"; reading A10). */
static uint32_t ko_mulhi(uint32_t w, uint32_t n) {
  return (uint32_t)(((uint64_t)w * (uint64_t)n) >> 32);
}

static int32_t ko_clamp(int64_t x, int32_t L) {
  if (x < 0) return 0;
  if (x > (int64_t)L - 1) return L - 1;
  return (int32_t)x;
}

/* ------------------------------------------------------------------------------------------
 * One agent's orders for (market m, step t, agent a) given the state at the start of the
 * step.  Returns the number of orders (1, or 2 for a maker); side 0 = bid (buy), 1 = ask
 * (sell).  Counter layout ctr = (agent, step, market, 0), key = (seed lo, seed hi).
 *   noise    buy = w0>>31; o = mulhi(w1, 2D+1) - D; q = 1 + mulhi(w2, qmax);
 *            tick = buy ? clamp(last - o) : clamp(last + o)           (reading A11)
 *   maker    s = 1 + mulhi(w1, spread_max); bid qty @ clamp(last - s) AND ask qty @
 *            clamp(last + s)                                          (reading A13)
 *   momentum dp = last - prev; buy = dp>0 ? 1 : dp<0 ? 0 : w0>>31; o = mulhi(w1, delta+1);
 *            q = 1 + mulhi(w2, qmax); tick = buy ? clamp(last + o) : clamp(last - o) (A12)
 * Type: model 0 -> all noise; model 1 -> a mod 3 = 0 noise, 1 maker, 2 momentum (A14).
 *
 * PACKED4 draw contract (models 2 = ZI rules, 3 = three types, DESIGN.md
 * reading A22): a separately named contract, NOT the BASELINE.json one.  One Philox block
 * serves four consecutive agents, w = Philox(ctr = (a >> 2, step, market, 0), key)[a & 3],
 * and every draw of the agent comes out of that one word by successive multiply-extract
 * (the high word of x*n is the draw, the low word is the still-unused randomness):
 *   noise    o = mulhi(w, 2D+1) - D, x1 = lo32(w*(2D+1)); q = 1 + mulhi(x1, qmax),
 *            x2 = lo32(x1*qmax); buy = x2>>31; tick as above
 *   maker    s = 1 + mulhi(w, spread_max); orders as above
 *   momentum o = mulhi(w, delta+1), x1 = lo32(w*(delta+1)); q = 1 + mulhi(x1, qmax),
 *            x2 = lo32(x1*qmax); buy = dp>0 ? 1 : dp<0 ? 0 : x2>>31; tick as above
 * Equivalently (exact integers): with N = n*qmax*2, J = floor(w*N / 2^32) and the draws
 * are J's mixed-radix digits, J = ((o_index*qmax) + (q-1))*2 + buy -- which is how the
 * pin in tests/test_oracle_packed.py checks them.
 * ---------------------------------------------------------------------------------------- */
static int32_t ko_gen_orders_packed4(const ko_params* P, int32_t L, int32_t last, int32_t prev,
                                     uint64_t seed, uint32_t m, uint32_t t, uint32_t a,
                                     int32_t side[2], int32_t tick[2], int32_t qty[2]) {
  uint32_t ctr[4] = { a >> 2, t, m, 0u };
  uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
  uint32_t out[4];
  ko_philox4x32_10(ctr, key, out);
  const uint32_t w = out[a & 3u];
  int type = 0;
  if (P->model == 3) type = (int)(a % 3u);
  if (type == 1) {
    int64_t s = 1 + (int64_t)ko_mulhi(w, (uint32_t)P->maker_spread_max);
    side[0] = 0; tick[0] = ko_clamp((int64_t)last - s, L); qty[0] = P->maker_qty;
    side[1] = 1; tick[1] = ko_clamp((int64_t)last + s, L); qty[1] = P->maker_qty;
    return 2;
  }
  const uint32_t n = type == 0 ? (uint32_t)(2 * P->noise_delta + 1) : (uint32_t)(P->mom_delta + 1);
  const uint32_t qmax = type == 0 ? (uint32_t)P->noise_qmax : (uint32_t)P->mom_qmax;
  const uint32_t oi = ko_mulhi(w, n);
  const uint32_t x1 = (uint32_t)((uint64_t)w * (uint64_t)n);
  const int32_t q = 1 + (int32_t)ko_mulhi(x1, qmax);
  const uint32_t x2 = (uint32_t)((uint64_t)x1 * (uint64_t)qmax);
  const int coin = (int)(x2 >> 31);
  if (type == 0) {
    int64_t o = (int64_t)oi - (int64_t)P->noise_delta;
    side[0] = coin ? 0 : 1;
    tick[0] = coin ? ko_clamp((int64_t)last - o, L) : ko_clamp((int64_t)last + o, L);
  } else {
    int64_t dp = (int64_t)last - (int64_t)prev;
    int buy = dp > 0 ? 1 : (dp < 0 ? 0 : coin);
    side[0] = buy ? 0 : 1;
    tick[0] = buy ? ko_clamp((int64_t)last + (int64_t)oi, L) : ko_clamp((int64_t)last - (int64_t)oi, L);
  }
  qty[0] = q;
  return 1;
}

/* ------------------------------------------------------------------------------------------
 * Model 4: the paper's own agent model (SIII-C; DESIGN.md
 * reading A24), in doubled-integer arithmetic so that no half-tick is ever rounded in floating
 * point.  State retrieval (Eq.3): bb = highest tick with resting bid depth, ba =
 * lowest tick with resting ask depth, at the start of the step;
 *     mid2 = 2*mid = bb + ba if both sides rest, else 2*last.
 * round(x) is round-half-up: round(m2/2) = floor((m2 + 1) / 2).  Classes by contiguous index
 * ranges (the paper gives class FRACTIONS): agents [0, A - n_mom - n_maker) noise,
 * then n_mom momentum, then n_maker makers.  Words of Philox(ctr = (a, t, m, 0)):
 *   w0>>31 coin; w1 -> eta; w2 -> quantity; w3>>16 < pmkt_q16 -> marketable.
 *   noise    buy = coin; eta = mulhi(w1, 2D+1) - D; p = round(mid + eta); q = 1 + mulhi(w2, qmax);
 *            marketable: p = L-1 for a buy, 0 for a sell
 *   momentum ret = sgn(mid2 - mid2_prev) (mid2_prev = doubled mid at the start of the previous
 *            step; 2*init before the first); buy = ret>0 ? 1 : ret<0 ? 0 : coin;
 *            p = round(mid + 1) for a buy, round(mid - 1) for a sell; q = 1 + mulhi(w2, mom_qmax);
 *            marketable like noise
 *   maker    buys if (a + t) mod 2 == 0 else sells; p = round(mid - h) for a bid, round(mid + h)
 *            for an ask, h = maker_spread_max ticks; q = 1 + mulhi(w2, maker_qty); never
 *            marketable
 * p is clamped to the grid (A15).  One order per agent.
 * ---------------------------------------------------------------------------------------- */
static int32_t ko_round_half_up(int64_t m2) {            /* floor((m2 + 1) / 2) for any sign */
  int64_t x = m2 + 1;
  return (int32_t)(x >= 0 ? x / 2 : -((-x + 1) / 2));
}

KO_API int32_t ko_gen_orders_paper(const ko_params* P, int32_t L, int32_t mid2, int32_t mid2_prev,
                                   uint64_t seed, uint32_t m, uint32_t t, uint32_t a, int32_t A,
                                   int32_t* side, int32_t* tick, int32_t* qty) {
  uint32_t ctr[4] = { a, t, m, 0u };
  uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
  uint32_t w[4];
  ko_philox4x32_10(ctr, key, w);
  const int32_t n_noise = A - P->paper_n_mom - P->paper_n_maker;
  const int coin = (int)(w[0] >> 31);
  const int mkt = (int32_t)(w[3] >> 16) < P->paper_pmkt_q16;
  int buy; int64_t p2; int32_t q; int can_mkt = 1;
  if ((int32_t)a < n_noise) {
    int64_t eta = (int64_t)ko_mulhi(w[1], (uint32_t)(2 * P->noise_delta + 1)) - (int64_t)P->noise_delta;
    buy = coin;
    p2 = (int64_t)mid2 + 2 * eta;
    q = 1 + (int32_t)ko_mulhi(w[2], (uint32_t)P->noise_qmax);
  } else if ((int32_t)a < n_noise + P->paper_n_mom) {
    int64_t d = (int64_t)mid2 - (int64_t)mid2_prev;
    buy = d > 0 ? 1 : (d < 0 ? 0 : coin);
    p2 = (int64_t)mid2 + (buy ? 2 : -2);
    q = 1 + (int32_t)ko_mulhi(w[2], (uint32_t)P->mom_qmax);
  } else {
    buy = ((a + t) & 1u) == 0u;
    p2 = (int64_t)mid2 + (buy ? -2 : 2) * (int64_t)P->maker_spread_max;
    q = 1 + (int32_t)ko_mulhi(w[2], (uint32_t)P->maker_qty);
    can_mkt = 0;
  }
  int32_t p = ko_clamp((int64_t)ko_round_half_up(p2), L);
  if (can_mkt && mkt) p = buy ? L - 1 : 0;
  *side = buy ? 0 : 1; *tick = p; *qty = q;
  return 1;
}

KO_API int32_t ko_gen_orders(const ko_params* P, int32_t L, int32_t last, int32_t prev,
                             uint64_t seed, uint32_t m, uint32_t t, uint32_t a,
                             int32_t side[2], int32_t tick[2], int32_t qty[2]) {
  if (P->model >= 2) return ko_gen_orders_packed4(P, L, last, prev, seed, m, t, a, side, tick, qty);
  uint32_t ctr[4] = { a, t, m, 0u };
  uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
  uint32_t w[4];
  ko_philox4x32_10(ctr, key, w);
  int type = 0;
  if (P->model == 1) type = (int)(a % 3u);
  if (type == 0) {
    int buy = (int)(w[0] >> 31);
    int64_t o = (int64_t)ko_mulhi(w[1], (uint32_t)(2 * P->noise_delta + 1)) - (int64_t)P->noise_delta;
    int32_t q = 1 + (int32_t)ko_mulhi(w[2], (uint32_t)P->noise_qmax);
    side[0] = buy ? 0 : 1;
    tick[0] = buy ? ko_clamp((int64_t)last - o, L) : ko_clamp((int64_t)last + o, L);
    qty[0] = q;
    return 1;
  } else if (type == 1) {
    int64_t s = 1 + (int64_t)ko_mulhi(w[1], (uint32_t)P->maker_spread_max);
    side[0] = 0; tick[0] = ko_clamp((int64_t)last - s, L); qty[0] = P->maker_qty;
    side[1] = 1; tick[1] = ko_clamp((int64_t)last + s, L); qty[1] = P->maker_qty;
    return 2;
  } else {
    int64_t dp = (int64_t)last - (int64_t)prev;
    int buy = dp > 0 ? 1 : (dp < 0 ? 0 : (int)(w[0] >> 31));
    int64_t o = (int64_t)ko_mulhi(w[1], (uint32_t)(P->mom_delta + 1));
    int32_t q = 1 + (int32_t)ko_mulhi(w[2], (uint32_t)P->mom_qmax);
    side[0] = buy ? 0 : 1;
    tick[0] = buy ? ko_clamp((int64_t)last + o, L) : ko_clamp((int64_t)last - o, L);
    qty[0] = q;
    return 1;
  }
}

/* ------------------------------------------------------------------------------------------
 * Uniform-price call-auction clearing of one combined book, in place.  Pure function of
 * (bid, ask); valid for any L >= 1 (the paper's worked example has L = 5).
 *   D[p] = sum_{q >= p} bid[q],  S[p] = sum_{q <= p} ask[q]                (Eq.1)
 *   V[p] = min(D[p], S[p]);  Vmax = max_p V[p];  p* = lowest p with V[p] = Vmax
 *                                                   (Eq.2; ties PAPER.md:194, 210)
 *   if Vmax > 0: price priority -- the highest bids and the lowest asks fill first
 *   (PAPER.md:343-348): the volume still unfilled when the allocation reaches tick p from
 *   above is Vmax - D[p+1], so bid[p] keeps min(bid[p], max(0, D[p] - Vmax)); symmetrically
 *   ask[p] keeps min(ask[p], max(0, S[p] - Vmax)).  (new_bid = BUY - traded_buy.)
 *   if Vmax = 0 nothing trades and the book is unchanged (reading A4).
 * D, S, V (each L int64, may be NULL) receive the profiles of the book BEFORE allocation.
 * *pstar = -1 when Vmax = 0.
 * ---------------------------------------------------------------------------------------- */
KO_API void ko_clear_step(int64_t* bid, int64_t* ask, int32_t L,
                          int64_t* D_out, int64_t* S_out, int64_t* V_out,
                          int32_t* pstar, int64_t* vmax) {
  int64_t* D = (int64_t*)malloc(sizeof(int64_t) * (size_t)L);
  int64_t* S = (int64_t*)malloc(sizeof(int64_t) * (size_t)L);
  int64_t acc = 0;
  for (int32_t p = L - 1; p >= 0; --p) { acc += bid[p]; D[p] = acc; }
  acc = 0;
  for (int32_t p = 0; p < L; ++p) { acc += ask[p]; S[p] = acc; }
  int64_t best = 0; int32_t best_p = -1;
  for (int32_t p = 0; p < L; ++p) {
    int64_t V = D[p] < S[p] ? D[p] : S[p];
    if (V_out) V_out[p] = V;
    if (V > best) { best = V; best_p = p; }        /* strict > keeps the lowest tick */
  }
  if (D_out) memcpy(D_out, D, sizeof(int64_t) * (size_t)L);
  if (S_out) memcpy(S_out, S, sizeof(int64_t) * (size_t)L);
  if (best > 0) {
    for (int32_t p = 0; p < L; ++p) {
      int64_t rb = D[p] - best; if (rb < 0) rb = 0; if (rb < bid[p]) bid[p] = rb;
      int64_t ra = S[p] - best; if (ra < 0) ra = 0; if (ra < ask[p]) ask[p] = ra;
    }
  }
  *pstar = best_p;
  *vmax = best;
  free(D); free(S);
}

/* record initialisation: empty accumulators, last = prev = init price (L/2 if < 0, A9),
 * FNV-1a offset basis for the trajectory hash. */
KO_API void ko_init_record(int64_t rec[16], int32_t L, int32_t init_price) {
  for (int i = 0; i < 16; ++i) rec[i] = 0;
  int32_t p0 = init_price < 0 ? L / 2 : init_price;
  rec[F_LAST] = p0; rec[F_PREV] = p0;
  rec[F_HASH] = (int64_t)0xcbf29ce484222325ull;
}

/* model 4: f[13] starts as the doubled opening price (the "previous mid") */
KO_API void ko_init_record_paper(int64_t rec[16], int32_t L, int32_t init_price) {
  ko_init_record(rec, L, init_price);
  rec[F_PREV] = 2 * rec[F_LAST];
}

/* ------------------------------------------------------------------------------------------
 * Run S steps of ONE market with global id m, continuing from (bid, ask, rec).
 * bid/ask are int64[L] (the oracle's book is 64-bit; ko_run_markets narrows it and checks).
 * Step t uses Philox step index t = rec[F_STEPS] (global), so run(S1); run(S2) == run(S1+S2).
 * Returns 0, or a negative code if an internal consistency assertion fails:
 *   -1 negative depth, -2 executed buy volume != executed sell volume != Vmax,
 *   -3 a per-side sum reached 2^31 (the library's int32 contract would overflow).
 * ---------------------------------------------------------------------------------------- */
static int32_t ko_run_market_impl(const ko_params* P, int32_t L, int32_t A, uint64_t seed,
                                  uint32_t m, int64_t S, int64_t* bid, int64_t* ask, int64_t rec[16],
                                  int32_t* trace) {
  for (int64_t s = 0; s < S; ++s) {
    int32_t last = (int32_t)rec[F_LAST], prev = (int32_t)rec[F_PREV];
    uint32_t t = (uint32_t)rec[F_STEPS];
    /* model 4: state retrieval (Eq.3) on the resting book; rec[F_PREV] holds the
     * doubled mid of the previous step instead of the previous price */
    int32_t mid2 = 2 * last;
    if (P->model == 4) {
      int32_t bb = -1, ba = L;
      for (int32_t p = 0; p < L; ++p) { if (bid[p] > 0) bb = p; }
      for (int32_t p = L - 1; p >= 0; --p) { if (ask[p] > 0) ba = p; }
      if (bb >= 0 && ba < L) mid2 = bb + ba;
    }
    /* 1. orders: every agent sees (last, prev) as they were at the start of the step */
    for (int32_t a = 0; a < A; ++a) {
      int32_t side[2], tick[2], qty[2];
      int32_t n = P->model == 4
                      ? ko_gen_orders_paper(P, L, mid2, prev, seed, m, t, (uint32_t)a, A, side, tick, qty)
                      : ko_gen_orders(P, L, last, prev, seed, m, t, (uint32_t)a, side, tick, qty);
      for (int32_t i = 0; i < n; ++i) {
        if (side[i] == 0) { bid[tick[i]] += qty[i]; rec[F_SUBBUY] += qty[i]; }
        else              { ask[tick[i]] += qty[i]; rec[F_SUBSELL] += qty[i]; }
        rec[F_NORDERS] += 1;
      }
    }
    /* 2-4. clear the combined book in place */
    int64_t before_b = 0, before_a = 0, after_b = 0, after_a = 0;
    for (int32_t p = 0; p < L; ++p) { before_b += bid[p]; before_a += ask[p]; }
    if (before_b >= (1ll << 31) || before_a >= (1ll << 31)) return -3;
    int32_t pstar; int64_t vmax;
    ko_clear_step(bid, ask, L, NULL, NULL, NULL, &pstar, &vmax);
    for (int32_t p = 0; p < L; ++p) {
      if (bid[p] < 0 || ask[p] < 0) return -1;
      after_b += bid[p]; after_a += ask[p];
    }
    if (before_b - after_b != vmax || before_a - after_a != vmax) return -2;
    /* 5. state and statistics */
    int64_t before = rec[F_LAST];
    rec[F_PREV] = P->model == 4 ? (int64_t)mid2 : rec[F_LAST];
    uint64_t x;
    if (vmax > 0) {
      rec[F_LAST] = pstar;
      rec[F_NTRADES] += 1;
      rec[F_SUMVOL] += vmax;
      rec[F_SUMPX] += pstar;
      rec[F_SUMPX2] += (int64_t)pstar * pstar;
      rec[F_SUMPXVOL] += (int64_t)pstar * vmax;
      x = ((uint64_t)vmax << 16) | (uint64_t)(uint32_t)pstar;
    } else {
      x = 0xFFFFull;
    }
    int64_t r = rec[F_LAST] - before;
    rec[F_SUMRET] += r;
    rec[F_SUMRET2] += r * r;
    rec[F_SUMRET3] += r * r * r;
    rec[F_SUMRET4] += r * r * r * r;
    uint64_t h = (uint64_t)rec[F_HASH];
    h = (h ^ x) * 0x100000001b3ull;
    rec[F_HASH] = (int64_t)h;
    rec[F_STEPS] += 1;
    /* per-step trace: the price after the step and the executed volume */
    if (trace) { trace[2 * s] = (int32_t)rec[F_LAST]; trace[2 * s + 1] = (int32_t)vmax; }
  }
  return 0;
}

KO_API int32_t ko_run_market(const ko_params* P, int32_t L, int32_t A, uint64_t seed,
                             uint32_t m, int64_t S, int64_t* bid, int64_t* ask, int64_t rec[16]) {
  return ko_run_market_impl(P, L, A, seed, m, S, bid, ask, rec, NULL);
}

/* Run S steps of n markets (global ids in ids[]) from the int32 state (books[n][2][L], side 0
 * = bid, 1 = ask; recs[n][16]) and write the state back.  Single-threaded loop. */
static int32_t ko_run_markets_impl(const ko_params* P, int32_t L, int32_t A, uint64_t seed,
                                   const uint32_t* ids, int32_t n, int64_t S,
                                   int32_t* books, int64_t* recs, int32_t* trace) {
  int64_t* bid = (int64_t*)malloc(sizeof(int64_t) * (size_t)L);
  int64_t* ask = (int64_t*)malloc(sizeof(int64_t) * (size_t)L);
  int32_t rc = 0;
  for (int32_t i = 0; i < n && rc == 0; ++i) {
    int32_t* b = books + (size_t)i * 2 * (size_t)L;
    for (int32_t p = 0; p < L; ++p) { bid[p] = b[p]; ask[p] = b[L + p]; }
    rc = ko_run_market_impl(P, L, A, seed, ids[i], S, bid, ask, recs + (size_t)i * 16,
                            trace ? trace + (size_t)i * 2 * (size_t)S : NULL);
    for (int32_t p = 0; p < L; ++p) { b[p] = (int32_t)bid[p]; b[L + p] = (int32_t)ask[p]; }
  }
  free(bid); free(ask);
  return rc;
}

KO_API int32_t ko_run_markets(const ko_params* P, int32_t L, int32_t A, uint64_t seed,
                              const uint32_t* ids, int32_t n, int64_t S,
                              int32_t* books, int64_t* recs) {
  return ko_run_markets_impl(P, L, A, seed, ids, n, S, books, recs, NULL);
}

/* The same, also recording trace[n][S][2] = (price after the step, executed volume Vmax) for the
 * S steps of this call (the paper "records the price returns"). */
KO_API int32_t ko_run_markets_traced(const ko_params* P, int32_t L, int32_t A, uint64_t seed,
                                     const uint32_t* ids, int32_t n, int64_t S,
                                     int32_t* books, int64_t* recs, int32_t* trace) {
  return ko_run_markets_impl(P, L, A, seed, ids, n, S, books, recs, trace);
}

/* ------------------------------------------------------------------------------------------
 * Return statistics of ONE market's trace[S][2] (SIV-J, Fig.7; DESIGN.md
 * reading A23), plain two-pass definitions in fp64.  Returns r_t = p_t - p_{t-1} between
 * consecutive traced steps, t = 1..S-1 (n = S-1 of them); x-bar = mean.
 *   out[0] volatility   = sqrt(m2), m2 = sum (r - rbar)^2 / n            ("std dev", Fig.7)
 *   out[1] excess kurt. = m4 / m2^2 - 3, m4 = sum (r - rbar)^4 / n       (NaN if m2 = 0)
 *   out[2] volume/step  = sum_t Vmax_t / S                               (all S steps)
 *   out[3] mean return  = rbar
 *   out[4 + k-1]     ACF_r(k)   = sum_{t=k+1..n} (r_t - rbar)(r_{t-k} - rbar) / sum_t (r_t - rbar)^2
 *   out[4 + K + k-1] ACF_|r|(k) = the same for x_t = |r_t|               k = 1..K (NaN if 0/0)
 * n < 1 -> everything but out[2] is NaN.
 * ---------------------------------------------------------------------------------------- */
KO_API void ko_trace_stats(const int32_t* trace, int64_t S, int32_t K, double* out) {
  double nan = 0.0; nan = nan / nan;
  const int64_t n = S - 1;
  double vsum = 0.0;
  for (int64_t t = 0; t < S; ++t) vsum += (double)trace[2 * t + 1];
  for (int32_t i = 0; i < 4 + 2 * K; ++i) out[i] = nan;
  out[2] = S > 0 ? vsum / (double)S : nan;
  if (n < 1) return;
  double* r = (double*)malloc(sizeof(double) * (size_t)n);
  double* a = (double*)malloc(sizeof(double) * (size_t)n);
  double rbar = 0.0, abar = 0.0;
  for (int64_t t = 0; t < n; ++t) {
    r[t] = (double)((int64_t)trace[2 * (t + 1)] - (int64_t)trace[2 * t]);
    a[t] = r[t] < 0 ? -r[t] : r[t];
    rbar += r[t]; abar += a[t];
  }
  rbar /= (double)n; abar /= (double)n;
  double m2 = 0.0, m4 = 0.0, a2 = 0.0;
  for (int64_t t = 0; t < n; ++t) {
    double d = r[t] - rbar, e = a[t] - abar;
    m2 += d * d; m4 += d * d * d * d; a2 += e * e;
  }
  out[0] = sqrt(m2 / (double)n);
  out[1] = m2 > 0 ? (m4 / (double)n) / ((m2 / (double)n) * (m2 / (double)n)) - 3.0 : nan;
  out[3] = rbar;
  for (int32_t k = 1; k <= K; ++k) {
    double cr = 0.0, ca = 0.0;
    for (int64_t t = k; t < n; ++t) { cr += (r[t] - rbar) * (r[t - k] - rbar); ca += (a[t] - abar) * (a[t - k] - abar); }
    out[4 + k - 1] = m2 > 0 ? cr / m2 : nan;
    out[4 + K + k - 1] = a2 > 0 ? ca / a2 : nan;
  }
  free(r); free(a);
}

/* fp64 statistics derived on the host from the integer record:
 * out = { mean_px, vwap, vol_per_step, ret_mean, ret_var, excess_kurtosis }.
 * A quantity whose denominator is zero is reported as NaN (0.0/0.0). */
KO_API void ko_derived(const int64_t rec[16], double out[6]) {
  double nan = 0.0; nan = nan / nan;
  double steps = (double)rec[F_STEPS], ntr = (double)rec[F_NTRADES], vol = (double)rec[F_SUMVOL];
  out[0] = ntr > 0 ? (double)rec[F_SUMPX] / ntr : nan;
  out[1] = vol > 0 ? (double)rec[F_SUMPXVOL] / vol : nan;
  out[2] = steps > 0 ? vol / steps : nan;
  if (steps > 0) {
    double mu = (double)rec[F_SUMRET] / steps;
    double var = (double)rec[F_SUMRET2] / steps - mu * mu;
    double m4 = ((double)rec[F_SUMRET4] - 4.0 * mu * (double)rec[F_SUMRET3]
                 + 6.0 * mu * mu * (double)rec[F_SUMRET2]) / steps - 3.0 * mu * mu * mu * mu;
    out[3] = mu; out[4] = var;
    out[5] = var > 0 ? m4 / (var * var) - 3.0 : nan;
  } else { out[3] = nan; out[4] = nan; out[5] = nan; }
}
