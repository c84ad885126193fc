// ks_microbench.cu -- libkineticsim_bench.so: the ablation entry point and the roofline
// microbenchmarks declared in include/kineticsim_bench.h.  A separate library from the product
// (libkineticsim.so, which never allocates device memory): these calls allocate a few bytes of
// device scratch for themselves and time their own kernels.
// (0) the launch-per-step ablation, through the product's public ks_run,
// (1) shared-memory atomic ceilings, (2) generation-only (Philox + rule) ceiling built from the
// library's own device templates, (3) raw IMAD.WIDE / LOP3 issue rates.
#include "../../include/kineticsim_bench.h"
#include "ks_device.cuh"

#include <cstdio>
#include <cstring>

namespace {

// ---- (1) shared-memory atomics ---------------------------------------------------------------
// MODE 0 distinct banks, 1 order-distribution pattern, 2 pattern + warp aggregation, 3 one address.
template <int MODE>
__global__ void smem_atomic_kernel(int L, int delta, int iters, int* out) {
  extern __shared__ int32_t sbook[];                      // [2][L]
  for (int i = threadIdx.x; i < 2 * L; i += blockDim.x) sbook[i] = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31;
  ks::BookRef bref; bref.ptr = sbook; bref.saddr = (uint32_t)__cvta_generic_to_shared(sbook);
  const uint32_t n = 2u * (uint32_t)delta + 1u;
  uint32_t x = (blockIdx.x * 1024u + threadIdx.x) * 2654435761u + 12345u;
  int sink = 0;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      int idx;
      if (MODE == 0) {
        idx = ((it * 8 + k) * 32 + lane) & (2 * L - 1);    // lane -> its own bank, all lanes distinct
      } else if (MODE == 3) {
        idx = (it * 8 + k) & (2 * L - 1);
      } else {
        x = x * 1664525u + 1013904223u;                    // LCG: RNG cost kept out of the measurement
        uint32_t o = __umulhi(x, n);
        idx = (int)((x & 1u) * (uint32_t)L) + L / 2 - delta + (int)o;
      }
      if (MODE == 2) ks::book_add<1>(bref, 4u * (uint32_t)idx, 1, sink);
      else           ks::book_add<0>(bref, 4u * (uint32_t)idx, 1, sink);
    }
  }
  __syncthreads();
  if (sbook[threadIdx.x & (2 * L - 1)] == 0x7fffffff) out[0] = sink;   // keep the atomics alive
}

// ---- (2) generation only ---------------------------------------------------------------------
template <int MODEL, bool PACKED>
__global__ void generate_only_kernel(const __grid_constant__ ks::KernelParams P, int* out) {
  const int tid = threadIdx.x, T = blockDim.x;
  const uint32_t market = P.market_base + blockIdx.x;
  const ks::MarketUniform mu = ks::market_uniform(P, market);
  const ks::GenPlan<MODEL> gplan = ks::gen_plan<MODEL>(PACKED ? (uint32_t)P.A >> 2 : (uint32_t)P.A, tid, T);
  ks::BookRef bref; bref.ptr = nullptr; bref.saddr = 0;
  int sink = 0;
  int last = P.L / 2, prev = P.L / 2;
  for (long long s = 0; s < P.S; ++s) {
    const ks::StepUniform u = ks::step_uniform(P, mu, (uint32_t)s);
    const ks::RuleCtx rc = ks::rule_ctx(P, bref, last, prev);
    ks::generate_step<MODEL, 2, PACKED>(P, bref, mu, u, rc, gplan, tid == 0, sink);
  }
  if (sink == 0x12345678) out[0] = sink;
}

// ---- (3) raw pipes ---------------------------------------------------------------------------
// KIND 0: IMAD.WIDE (with accumulate); 1: LOP3; 2: one IMAD.WIDE + one dependent LOP3 (the Philox
// round pattern); 3, 4: one IMAD.WIDE + two / three LOP3 -- how much every further alu-pipe
// instruction costs the multiply stream.
template <int KIND>
__global__ void int_pipe_kernel(int iters, uint32_t seed, uint32_t* out) {
  uint32_t c[8], d[8], e[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) { c[j] = seed + threadIdx.x * 8u + j; d[j] = c[j] ^ 0x9E3779B9u; e[j] = d[j] * 3u; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (KIND == 0 || KIND == 2) {
          uint64_t p = (uint64_t)ks::kPhiloxM0 * c[j] + (((uint64_t)d[j] << 32) | c[j]);   // IMAD.WIDE.U32 with accumulate
          c[j] = (uint32_t)p; d[j] = (uint32_t)(p >> 32);
        }
        if (KIND == 1 || KIND == 2) {
          c[j] = c[j] ^ d[j] ^ seed;                                                       // LOP3
          if (KIND == 1) d[j] = d[j] ^ c[j] ^ 0x85EBCA6Bu;
        }
        if (KIND >= 3) {
          const uint64_t p = (uint64_t)ks::kPhiloxM0 * c[j];
          const uint32_t hi = (uint32_t)(p >> 32), lo = (uint32_t)p;
          c[j] = hi ^ d[j] ^ seed; d[j] = lo;                                              // LOP3 #1
          e[j] = e[j] ^ lo ^ seed;                                                         // LOP3 #2
          if (KIND == 4) e[j] = (e[j] & hi) ^ seed;                                        // LOP3 #3
        }
      }
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) acc ^= c[j] ^ d[j] ^ e[j];
  if (acc == 0x12345678u) out[0] = acc;
}

// KIND 5: a pure stream of mul.wide.u32 (IMAD.WIDE.U32 with no addend), 8 independent chains per
// thread, each feeding the high word of its product back in -- nothing but 32x32->64 multiplies
// on the fmaheavy pipe: the MEASURED peak the hot loop's multiplies are reported against.
__global__ void mul_wide_kernel(int iters, uint32_t seed, uint32_t* out) {
  uint32_t c[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) c[j] = seed + threadIdx.x * 8u + j;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        uint64_t p;
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(c[j]), "r"(ks::kPhiloxM0));
        c[j] = (uint32_t)(p >> 32);
      }
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) acc ^= c[j];
  if (acc == 0x12345678u) out[0] = acc;
}

template <typename F>
ks_status time_best(F launch, int warmup, int reps, cudaStream_t st, double* seconds) {
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return KS_ERR_CUDA;
  for (int i = 0; i < warmup; ++i) launch();
  float best = 1e30f;
  ks_status rc = KS_OK;
  for (int i = 0; i < reps; ++i) {
    cudaEventRecord(e0, st);
    launch();
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = KS_ERR_CUDA; break; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *seconds = best * 1e-3;
  return rc;
}

int num_sms() {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
  return sms;
}

}  // namespace

extern "C" {

// a8 ablation: the product's own ks_run, one launch per step, book through HBM between launches.
ks_status ks_run_stepwise(ks_sim* s, int64_t S, void* stream) {
  if (!s || S < 0) return KS_ERR_INVALID_ARG;
  for (int64_t i = 0; i < S; ++i) {
    ks_status r = ks_run(s, 1, stream);
    if (r != KS_OK) return r;
  }
  return KS_OK;
}

ks_status ks_bench_smem_atomic(int32_t mode, int32_t delta, int32_t L, int32_t threads, int32_t ctas_per_sm,
                               int32_t iters, int32_t warmup, int32_t reps, void* stream, double* lane_ops_per_s,
                               double* seconds) {
  if (!lane_ops_per_s || !seconds || mode < 0 || mode > 3 || L < 32 || (L & (L - 1)) || L > 8192 || delta < 0 ||
      2 * delta + 1 > L || threads < 32 || threads > 1024 || threads % 32 || ctas_per_sm < 1 || iters < 1 || reps < 1)
    return KS_ERR_INVALID_ARG;
  const int sms = num_sms();
  if (sms <= 0) return KS_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  int* d_out = nullptr;   // tiny scratch for the (never taken) sink store: a benchmark-only allocation
  if (cudaMalloc(&d_out, 64) != cudaSuccess) return KS_ERR_CUDA;
  const int grid = sms * ctas_per_sm;
  const size_t smem = (size_t)8 * L;
  auto launch = [&]() {
    switch (mode) {
      case 0: smem_atomic_kernel<0><<<grid, threads, smem, st>>>(L, delta, iters, d_out); break;
      case 1: smem_atomic_kernel<1><<<grid, threads, smem, st>>>(L, delta, iters, d_out); break;
      case 2: smem_atomic_kernel<2><<<grid, threads, smem, st>>>(L, delta, iters, d_out); break;
      default: smem_atomic_kernel<3><<<grid, threads, smem, st>>>(L, delta, iters, d_out); break;
    }
  };
  if (smem > 48 * 1024) {
    cudaFuncSetAttribute(smem_atomic_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(smem_atomic_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(smem_atomic_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(smem_atomic_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  ks_status rc = time_best(launch, warmup, reps, st, seconds);
  cudaFree(d_out);
  if (rc != KS_OK) return rc;
  *lane_ops_per_s = (double)grid * threads * (double)iters * 8.0 / *seconds;
  return KS_OK;
}

ks_status ks_bench_generate_only(const ks_agent_params* p, int32_t M, int32_t L, int32_t A, int64_t S, int32_t threads,
                                 int32_t warmup, int32_t reps, void* stream, double* events_per_s, double* seconds) {
  if (!p || !events_per_s || !seconds || M < 1 || L < 32 || (L & (L - 1)) || A < 0 || S < 1 || threads < 32 ||
      threads > 1024 || threads % 32 || reps < 1)
    return KS_ERR_INVALID_ARG;
  ks::KernelParams P;
  memset(&P, 0, sizeof(P));
  uint32_t k0 = 0x243F6A88u, k1 = 0x85A308D3u;
  for (int r = 0; r < 10; ++r) { P.k0[r] = k0; P.k1[r] = k1; k0 += ks::kPhiloxW0; k1 += ks::kPhiloxW1; }
  P.M = M; P.L = L; P.A = A; P.S = S;
  P.noise_delta = p->noise_delta; P.noise_n = 2 * p->noise_delta + 1; P.noise_qmax = p->noise_qmax;
  P.noise_n4 = 4 * P.noise_n; P.q_addend = 1ull << 32;
  P.maker_spread_max = p->maker_spread_max; P.maker_qty = p->maker_qty;
  P.mom_n = p->mom_delta + 1; P.mom_qmax = p->mom_qmax;
  const size_t smem = 0;
  cudaStream_t st = (cudaStream_t)stream;
  int* d_out = nullptr;
  if (cudaMalloc(&d_out, 64) != cudaSuccess) return KS_ERR_CUDA;
  const int model = p->model & 1, packed = p->model >> 1;
  auto launch = [&]() {
    if (model == 0) {
      if (packed) generate_only_kernel<0, true><<<M, threads, smem, st>>>(P, d_out);
      else        generate_only_kernel<0, false><<<M, threads, smem, st>>>(P, d_out);
    } else {
      if (packed) generate_only_kernel<1, true><<<M, threads, smem, st>>>(P, d_out);
      else        generate_only_kernel<1, false><<<M, threads, smem, st>>>(P, d_out);
    }
  };
  ks_status rc = time_best(launch, warmup, reps, st, seconds);
  cudaFree(d_out);
  if (rc != KS_OK) return rc;
  *events_per_s = (double)M * (double)A * (double)S / *seconds;
  return KS_OK;
}

ks_status ks_bench_int_pipe(int32_t kind, int32_t threads, int32_t ctas_per_sm, int32_t iters, int32_t warmup,
                            int32_t reps, void* stream, double* thread_ops_per_s, double* seconds) {
  if (!thread_ops_per_s || !seconds || kind < 0 || kind > 5 || threads < 32 || threads > 1024 || threads % 32 ||
      ctas_per_sm < 1 || iters < 1 || reps < 1)
    return KS_ERR_INVALID_ARG;
  const int sms = num_sms();
  if (sms <= 0) return KS_ERR_CUDA;
  cudaStream_t st = (cudaStream_t)stream;
  uint32_t* d_out = nullptr;
  if (cudaMalloc(&d_out, 64) != cudaSuccess) return KS_ERR_CUDA;
  const int grid = sms * ctas_per_sm;
  auto launch = [&]() {
    if (kind == 0)      int_pipe_kernel<0><<<grid, threads, 0, st>>>(iters, 7u, d_out);
    else if (kind == 1) int_pipe_kernel<1><<<grid, threads, 0, st>>>(iters, 7u, d_out);
    else if (kind == 2) int_pipe_kernel<2><<<grid, threads, 0, st>>>(iters, 7u, d_out);
    else if (kind == 3) int_pipe_kernel<3><<<grid, threads, 0, st>>>(iters, 7u, d_out);
    else if (kind == 4) int_pipe_kernel<4><<<grid, threads, 0, st>>>(iters, 7u, d_out);
    else                mul_wide_kernel<<<grid, threads, 0, st>>>(iters, 7u, d_out);
  };
  ks_status rc = time_best(launch, warmup, reps, st, seconds);
  cudaFree(d_out);
  if (rc != KS_OK) return rc;
  const double per_iter = (kind == 0 || kind == 5 ? 1.0 : (kind <= 2 ? 2.0 : (kind == 3 ? 3.0 : 4.0))) * 32.0;   // ops per thread per iteration
  *thread_ops_per_s = (double)grid * threads * (double)iters * per_iter / *seconds;
  return KS_OK;
}

}  // extern "C"
