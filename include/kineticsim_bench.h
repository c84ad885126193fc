/*
 * kineticsim_bench.h -- ablation and roofline-microbenchmark entry points, exported by a SEPARATE
 * library (libkineticsim_bench.so, linked against libkineticsim.so).  Not part of the product ABI
 * (include/kineticsim.h); used by bench.py, the tests and DESIGN.md's measurement section.  Same
 * conventions as kineticsim.h, except that the ks_bench_* calls allocate a few bytes of device
 * scratch for themselves (the product library never allocates device memory) and are SYNCHRONOUS:
 * they time their own kernel with CUDA events on `stream` (after `warmup` untimed launches) and
 * return the best of `reps` timed launches.
 */
#ifndef KINETICSIM_BENCH_H_
#define KINETICSIM_BENCH_H_

#include "kineticsim.h"

#ifdef __cplusplus
extern "C" {
#endif

/* a8 ablation (SIII-F "naive" traffic): the same step as ks_run, but ONE LAUNCH
 * PER STEP with the book stored to and re-loaded from HBM between launches, so global traffic is
 * Theta(S*M*L) instead of Theta(M*L).  Leaves bit-identical state to ks_run(S).  Implemented as S
 * calls of the product's public ks_run(s, 1, stream). */
KS_API ks_status ks_run_stepwise(ks_sim* s, int64_t S, void* stream);

/* Shared-memory atomic ceilings (BASELINE.json `metric`: "% of smem-atomic roofline").
 * Every SM runs `ctas_per_sm` CTAs of `threads` threads; each lane issues `iters` x 8 independent
 * int32 atomicAdd (result unused -> ATOMS.ADD) into a CTA-private shared array.
 *   mode 0  peak: lane i of every warp hits its own bank, no two lanes share an address
 *   mode 1  pattern: side and tick drawn by a 1-multiply LCG with the order distribution of a
 *           zero-intelligence config: 2 sides x (2*delta+1) ticks around L/2 in a [2][L] book
 *   mode 2  pattern, warp-aggregated with __match_any_sync / __reduce_add_sync before the atomic
 *   mode 3  worst case: all 32 lanes hit one address
 * *lane_ops_per_s receives atomic lane-operations per second (orders/s a kernel doing nothing
 * but the atomics could aggregate). */
KS_API ks_status ks_bench_smem_atomic(int32_t mode, int32_t delta, int32_t L, int32_t threads,
                                      int32_t ctas_per_sm, int32_t iters, int32_t warmup, int32_t reps,
                                      void* stream, double* lane_ops_per_s, double* seconds);

/* Integer-ALU ceiling for this RNG contract: the library's own generation code (Philox4x32-10 +
 * agent rule, same templates as the persistent kernel) with the shared-memory atomic replaced by
 * a register fold.  Runs M CTAs x `threads` threads, S steps of A agents with a fixed price.
 * *events_per_s receives agent events per second. */
KS_API ks_status ks_bench_generate_only(const ks_agent_params* p, int32_t M, int32_t L, int32_t A, int64_t S,
                                        int32_t threads, int32_t warmup, int32_t reps,
                                        void* stream, double* events_per_s, double* seconds);

/* Raw issue rates of the two instructions Philox is made of.  kind 0: IMAD.WIDE.U32 (u32 x u32 ->
 * u64), kind 1: LOP3 (three-input xor), kind 2: one of each, interleaved (the Philox round
 * pattern), kind 3 / 4: one IMAD.WIDE with two / three LOP3 (what every further alu-pipe instruction
 * costs the multiply stream), kind 5: a pure stream of mul.wide.u32 with no addend (IMAD.WIDE.U32
 * only) -- the measured peak of the pipe that bounds the hot loop (roofline.peak in bench.py).
 * Each thread runs 8 independent dependency chains.  *thread_ops_per_s receives thread-level operations per second
 * over the whole GPU (divide by 32 x SMs x 4 x clock for warp instructions per cycle per
 * scheduler). */
KS_API ks_status ks_bench_int_pipe(int32_t kind, int32_t threads, int32_t ctas_per_sm, int32_t iters,
                                   int32_t warmup, int32_t reps, void* stream, double* thread_ops_per_s,
                                   double* seconds);

#ifdef __cplusplus
}
#endif
#endif /* KINETICSIM_BENCH_H_ */
