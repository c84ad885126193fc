// ks_api.cu -- host side of the C ABI declared in include/kineticsim.h.
#include "../../include/kineticsim.h"
#include "ks_cluster.cuh"
#include "ks_decoupled.cuh"
#include "ks_trace.cuh"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

namespace {

thread_local char g_err[512] = "";
std::atomic<long long> g_launches{0};

void set_err(const char* fmt, const char* a = "", const char* b = "") {
  snprintf(g_err, sizeof(g_err), fmt, a, b);
}

#define KS_CUDA(call)                                                 \
  do {                                                                \
    cudaError_t e_ = (call);                                          \
    if (e_ != cudaSuccess) {                                          \
      set_err("%s failed: %s", #call, cudaGetErrorString(e_));        \
      return KS_ERR_CUDA;                                             \
    }                                                                 \
  } while (0)

bool is_pow2(int32_t x) { return x > 0 && (x & (x - 1)) == 0; }

constexpr int32_t kMaxLPerCta = 16384;    // 8*Lc = 128 KB of the 227 KB a CTA may own
constexpr int32_t kMaxL = 32768;          // p* must fit the 16-bit field of the trajectory hash
constexpr int32_t kMaxQty = 1 << 20;

}  // namespace

struct ks_sim {
  int32_t M, L, A;
  ks_agent_params p;
  uint64_t seed;
  uint32_t market_base;
  void* d_state;
  int64_t steps_done;
  int64_t resting_bound;      // bound on the per-side depth total injected by ks_write_books / found by ks_attach
  int32_t fresh;              // books known all-zero (no run, no ks_write_books yet)
  int32_t opt_threads, opt_atomic, opt_clear, opt_cluster, opt_pipe, opt_cols, opt_ring, opt_pair;
  int32_t n_noise, n_maker, n_mom;
  int64_t inflow_per_step;    // per-side bound on the quantity one step can add
  unsigned long long* h_words;   // pinned, mapped host memory: [0] depth bound of ks_write_books (copied),
                                 // [1] sticky error flags written by the kernels themselves (ks::kFlag*)
  unsigned long long* d_flags;   // device alias of &h_words[1]
  cudaEvent_t bound_event;
  int32_t bound_pending;         // a ks_write_books depth check whose result the host has not seen yet
  int32_t dev_smem_optin;
  int32_t num_sms;
  int32_t device;                // the CUDA device d_state lives on (the current one at creation)
};

namespace {

// Makes the handle's device current for the duration of a call (a process may hold several GPUs).
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// Sticky device-raised errors.  The kernels write them into mapped host memory; a caller that can
// see a run's results has synchronised the stream and therefore cannot miss the flag.
ks_status check_flags(const ks_sim* s, const char* who) {
  const unsigned long long f = *reinterpret_cast<volatile unsigned long long*>(&s->h_words[1]);
  if (f == 0) return KS_OK;
  if (f & ks::kFlagNegativeDepth) { set_err("%s: ks_write_books stored a negative depth; the following run was not executed", who); return KS_ERR_INVALID_ARG; }
  if (f & ks::kFlagDepthOverflow) { set_err("%s: per-side depth could reach 2^31; the run was not executed", who); return KS_ERR_OVERFLOW; }
  set_err("%s: a statistic (sum of r^3 or r^4) left int64 during an earlier run", who);
  return KS_ERR_OVERFLOW;
}

int32_t* books_ptr(const ks_sim* s) { return reinterpret_cast<int32_t*>(s->d_state); }
long long* recs_ptr(const ks_sim* s) {
  return reinterpret_cast<long long*>(reinterpret_cast<char*>(s->d_state) + (size_t)s->M * 8 * (size_t)s->L);
}
unsigned long long* scratch_ptr(const ks_sim* s) {
  return reinterpret_cast<unsigned long long*>(reinterpret_cast<char*>(s->d_state) +
                                               (size_t)s->M * (8 * (size_t)s->L + 128));
}

bool shape_ok(int32_t M, int32_t L) { return M >= 1 && is_pow2(L) && L >= 32 && L <= 32768; }

void free_sim(ks_sim* s) {
  if (!s) return;
  if (s->h_words) cudaFreeHost(s->h_words);
  if (s->bound_event) cudaEventDestroy(s->bound_event);
  delete s;
}

// Enqueue the depth check of the books in d_state: max over markets and sides of the total depth
// -> scratch word -> h_words[0]; bound_event marks its completion.
ks_status enqueue_depth_check(ks_sim* s, cudaStream_t st) {
  KS_CUDA(cudaMemsetAsync(scratch_ptr(s), 0, sizeof(unsigned long long), st));
  ks::ks_depth_bound_kernel<<<2 * s->M, 128, 0, st>>>(books_ptr(s), s->L, scratch_ptr(s));
  KS_CUDA(cudaGetLastError());
  g_launches++;
  KS_CUDA(cudaMemcpyAsync(&s->h_words[0], scratch_ptr(s), sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  KS_CUDA(cudaEventRecord(s->bound_event, st));
  s->bound_pending = 1;
  return KS_OK;
}

// ks_create_ex (attach = false: enqueue the initialisation) and ks_attach (attach = true: adopt
// the state already in d_state).
ks_status create_common(ks_sim** out, int32_t M, int32_t L, int32_t A, const ks_agent_params* p, uint64_t seed,
                        uint32_t market_base, void* d_state, void* stream, bool attach) {
  const char* who = attach ? "ks_attach" : "ks_create";
  if (!out || !p || !d_state) { set_err("%s: NULL argument", who); return KS_ERR_INVALID_ARG; }
  *out = nullptr;
  if (M < 1 || A < 0 || !is_pow2(L) || L < 32) { set_err("%s: need M >= 1, A >= 0, L a power of two >= 32", who); return KS_ERR_INVALID_ARG; }
  if (L > kMaxL) { set_err("%s: L > 32768 is not supported (p* must fit 16 bits of the trajectory hash)", who); return KS_ERR_UNSUPPORTED; }
  if ((reinterpret_cast<uintptr_t>(d_state) & 15) != 0) { set_err("%s: d_state must be 16-byte aligned", who); return KS_ERR_INVALID_ARG; }
  if (p->model < KS_MODEL_ZI || p->model > KS_MODEL_PAPER) { set_err("%s: unknown model", who); return KS_ERR_INVALID_ARG; }
  if (p->noise_delta < 0 || p->noise_delta >= L || p->noise_qmax < 1 || p->noise_qmax > kMaxQty || p->init_price >= L) {
    set_err("%s: bad noise parameters or init_price", who); return KS_ERR_INVALID_ARG;
  }
  if (p->model == KS_MODEL_PAPER) {
    if (p->maker_spread_max < 0 || p->maker_spread_max >= L || p->maker_qty < 1 || p->maker_qty > kMaxQty ||
        p->mom_qmax < 1 || p->mom_qmax > kMaxQty || p->paper_n_mom < 0 || p->paper_n_maker < 0 ||
        (int64_t)p->paper_n_mom + p->paper_n_maker > A || p->paper_pmkt_q16 < 0 || p->paper_pmkt_q16 > 65536) {
      set_err("%s: bad parameters of the paper agent model", who); return KS_ERR_INVALID_ARG;
    }
    if (L > kMaxLPerCta) { set_err("%s: the paper agent model has no cluster path (L <= 16384)", who); return KS_ERR_UNSUPPORTED; }
  } else if ((p->model & 1) == KS_MODEL_MIX3 &&
      (p->maker_spread_max < 1 || p->maker_spread_max > L || p->maker_qty < 1 || p->maker_qty > kMaxQty ||
       p->mom_delta < 0 || p->mom_delta >= L || p->mom_qmax < 1 || p->mom_qmax > kMaxQty)) {
    set_err("%s: bad maker/momentum parameters", who); return KS_ERR_INVALID_ARG;
  }
  if ((uint64_t)market_base + (uint64_t)M > 0x100000000ull) { set_err("%s: market ids exceed 32 bits", who); return KS_ERR_INVALID_ARG; }

  int dev = 0, optin = 0, sms = 0;
  KS_CUDA(cudaGetDevice(&dev));
  KS_CUDA(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  KS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  {
    const int32_t Lc = L > kMaxLPerCta ? kMaxLPerCta : L;           // larger books are split across a cluster
    if ((size_t)8 * Lc + 2048 > (size_t)optin) { set_err("%s: book does not fit this device's shared memory", who); return KS_ERR_UNSUPPORTED; }
  }

  ks_sim* s = new (std::nothrow) ks_sim();
  if (!s) { set_err("%s: out of host memory", who); return KS_ERR_NOMEM; }
  s->M = M; s->L = L; s->A = A; s->p = *p; s->seed = seed; s->market_base = market_base;
  s->d_state = d_state; s->steps_done = 0; s->resting_bound = 0; s->fresh = attach ? 0 : 1;
  s->opt_threads = 0; s->opt_atomic = 0; s->opt_clear = 0; s->opt_cluster = 0; s->opt_pipe = 0; s->opt_cols = 0; s->opt_ring = 0; s->opt_pair = 0;
  s->dev_smem_optin = optin; s->num_sms = sms; s->device = dev;
  s->bound_pending = 0; s->h_words = nullptr; s->d_flags = nullptr; s->bound_event = nullptr;
  if (p->model == KS_MODEL_PAPER) {
    s->n_mom = p->paper_n_mom; s->n_maker = 0; s->n_noise = A - p->paper_n_mom - p->paper_n_maker;
    s->inflow_per_step = (int64_t)s->n_noise * p->noise_qmax + (int64_t)p->paper_n_mom * p->mom_qmax +
                         (int64_t)p->paper_n_maker * p->maker_qty;
  } else if ((p->model & 1) == KS_MODEL_ZI) {
    s->n_noise = A; s->n_maker = 0; s->n_mom = 0;
    s->inflow_per_step = (int64_t)A * p->noise_qmax;
  } else {
    s->n_noise = (A + 2) / 3; s->n_maker = (A + 1) / 3; s->n_mom = A / 3;
    s->inflow_per_step = (int64_t)s->n_noise * p->noise_qmax + (int64_t)s->n_maker * p->maker_qty +
                         (int64_t)s->n_mom * p->mom_qmax;
  }
  if (s->p.init_price < 0) s->p.init_price = L / 2;

  cudaError_t e = cudaHostAlloc(reinterpret_cast<void**>(&s->h_words), 2 * sizeof(unsigned long long), cudaHostAllocMapped);
  if (e == cudaSuccess) { s->h_words[0] = 0; s->h_words[1] = 0; }
  if (e == cudaSuccess) {
    void* dp = nullptr;
    e = cudaHostGetDevicePointer(&dp, &s->h_words[1], 0);
    s->d_flags = reinterpret_cast<unsigned long long*>(dp);
  }
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->bound_event, cudaEventDisableTiming);
  if (e != cudaSuccess) {
    set_err("%s: %s", who, cudaGetErrorString(e));
    free_sim(s);
    return KS_ERR_CUDA;
  }

  cudaStream_t st = (cudaStream_t)stream;
  if (!attach) {
    size_t nvec = (size_t)M * 2 * (size_t)L / 4;
    int blocks = (int)((nvec + 255) / 256);
    if (blocks > sms * 16) blocks = sms * 16;
    if (blocks < 1) blocks = 1;
    ks::ks_init_kernel<<<blocks, 256, 0, st>>>(reinterpret_cast<int4*>(books_ptr(s)), nvec, recs_ptr(s), M, s->p.init_price,
                                               p->model == KS_MODEL_PAPER ? 2 * s->p.init_price : s->p.init_price);
    e = cudaGetLastError();
    if (e != cudaSuccess) {
      set_err("%s: init launch failed: %s", who, cudaGetErrorString(e));
      free_sim(s);
      return KS_ERR_CUDA;
    }
    g_launches++;
  } else {
    // adopt the checkpoint: the step counter (for the overflow guards) and the resting depth bound
    // come back from the device; this call synchronises `stream`
    // scratch words [1] = largest step counter over the markets, [2] = 1 when some record cannot be
    // one this library wrote (negative step counter, price off the grid)
    unsigned long long chk[2] = {0, 0};
    long long steps0 = 0;
    ks_status r = enqueue_depth_check(s, st);
    if (r == KS_OK) {
      e = cudaMemsetAsync(scratch_ptr(s) + 1, 0, 2 * sizeof(unsigned long long), st);
      if (e == cudaSuccess) {
        ks::ks_attach_check_kernel<<<(M + 255) / 256, 256, 0, st>>>(recs_ptr(s), M, L, p->model == KS_MODEL_PAPER ? 2 * L - 1 : L,
                                                                    scratch_ptr(s) + 1);
        e = cudaGetLastError();
        if (e == cudaSuccess) g_launches++;
      }
      if (e == cudaSuccess) e = cudaMemcpyAsync(chk, scratch_ptr(s) + 1, sizeof(chk), cudaMemcpyDeviceToHost, st);
      if (e == cudaSuccess) e = cudaStreamSynchronize(st);
      if (e != cudaSuccess) { set_err("%s: %s", who, cudaGetErrorString(e)); r = KS_ERR_CUDA; }
      steps0 = (long long)chk[0];
    }
    if (r == KS_OK && chk[1] != 0) { set_err("%s: d_state does not hold valid records (a negative step counter or a price off the grid)", who); r = KS_ERR_INVALID_ARG; }
    if (r == KS_OK && (steps0 < 0 || steps0 >= 4294967296LL)) { set_err("%s: d_state does not hold a valid record (step counter)", who); r = KS_ERR_INVALID_ARG; }
    if (r == KS_OK && s->h_words[0] == 0xffffffffffffffffull) { set_err("%s: d_state holds a negative depth", who); r = KS_ERR_INVALID_ARG; }
    if (r != KS_OK) { free_sim(s); return r; }
    s->bound_pending = 0;
    s->steps_done = steps0;
    s->resting_bound = (int64_t)s->h_words[0];
  }
  *out = s;
  return KS_OK;
}

}  // namespace

extern "C" {

size_t ks_state_bytes(int32_t M, int32_t L) {
  if (!shape_ok(M, L)) return 0;
  return (size_t)M * (8 * (size_t)L + 128) + 256;
}

const char* ks_last_error(void) { return g_err; }
int64_t ks_launch_count(void) { return g_launches.load(); }

ks_status ks_create(ks_sim** out, int32_t M, int32_t L, int32_t A, const ks_agent_params* p, uint64_t seed,
                    void* d_state, void* stream) {
  return create_common(out, M, L, A, p, seed, 0u, d_state, stream, false);
}

ks_status ks_create_ex(ks_sim** out, int32_t M, int32_t L, int32_t A, const ks_agent_params* p, uint64_t seed,
                       uint32_t market_base, void* d_state, void* stream) {
  return create_common(out, M, L, A, p, seed, market_base, d_state, stream, false);
}

ks_status ks_attach(ks_sim** out, int32_t M, int32_t L, int32_t A, const ks_agent_params* p, uint64_t seed,
                    uint32_t market_base, void* d_state, void* stream) {
  return create_common(out, M, L, A, p, seed, market_base, d_state, stream, true);
}

void ks_destroy(ks_sim* s) {
  if (!s) return;
  DeviceGuard g(s->device);
  free_sim(s);
}

ks_status ks_set_option(ks_sim* s, int32_t option, int32_t value) {
  if (!s) { set_err("ks_set_option: NULL handle"); return KS_ERR_INVALID_ARG; }
  switch (option) {
    case KS_OPT_BLOCK_THREADS:
      if (value != 0 && (value < 32 || value > 1024 || value % 32 != 0)) break;
      s->opt_threads = value; return KS_OK;
    case KS_OPT_ATOMIC_MODE:
      if (value != 0 && value != 1) break;
      if (value == 1 && (s->opt_cluster > 1 || s->L > kMaxLPerCta)) break;   // the cluster kernel has plain atomics only
      if (value == 1 && s->p.model >= KS_MODEL_ZI_PACKED4) break;            // so have PACKED4 and the paper model
      s->opt_atomic = value; return KS_OK;
    case KS_OPT_CLEAR_PATH:
      if (value != 0 && value != 1) break;
      s->opt_clear = value; return KS_OK;
    case KS_OPT_PIPELINE:
      if (value != 0 && value != 1 && value != 2) break;
      s->opt_pipe = value; return KS_OK;
    case KS_OPT_REL_COLUMNS:
      if (value != 0 && value != 1) break;
      s->opt_cols = value; return KS_OK;
    case KS_OPT_STEP_PAIRS:
      if (value != 0 && value != 1 && value != 2) break;
      s->opt_pair = value; return KS_OK;
    case KS_OPT_RING_DEPTH:
      if (value != 0 && value != 2 && value != 4) break;
      s->opt_ring = value; return KS_OK;
    case KS_OPT_CLUSTER_SIZE:
      if (value != 0 && value != 1 && value != 2 && value != 4 && value != 8) break;
      if (value > 1 && (s->L / value < 32 || s->opt_atomic || s->p.model == KS_MODEL_PAPER)) break;
      if (value == 1 && s->L > kMaxLPerCta) break;
      s->opt_cluster = value; return KS_OK;
    default: break;
  }
  set_err("ks_set_option: unknown option or value");
  return KS_ERR_INVALID_ARG;
}

}  // extern "C"

// Launch plan: threads per CTA and dynamic shared memory (the book).  An SM has 228 KB of shared
// memory; each resident CTA costs its dynamic + static allocation + 1 KB of system reserve, and an
// SM holds at most 32 CTAs.
// Threads: many markets and a small book -> ONE WARP per market (T = 32, 32 CTAs per SM): no warp
// ever waits at a barrier for another warp's generation or for the clearing warp, and the eight
// markets resident on a scheduler hide each other's clearing (measured on B200, DESIGN.md 7.4:
// T = 32 beats 64/128 on C4).  A book so large that 32-thread CTAs would leave the SM short of
// warps -> widen until ~1024 threads are resident; few markets -> widen so the whole GPU is used,
// but never beyond the agents.
struct LaunchPlan { int T; size_t smem; bool decoupled; uint32_t rel_side; int ring; int group; bool mix; uint32_t rel_stride, mk_off, mom_off, mom_side; };

static const long long kSmemPerSM = 228LL * 1024, kSmemCtaOverhead = 1024 + 1024;   // reserve + static

// Bytes of one side (sell or buy bins) of one relative histogram of ks_decoupled_kernel: 2*delta+1
// bins of one int32 (padded to 128 bytes) or of 32 lane columns.  One buffer = two sides.
static uint32_t rel_side_for(const ks_sim* s) {
  const uint32_t n = 2u * (uint32_t)s->p.noise_delta + 1u;
  return s->opt_cols ? n * 128u : ((n * 4u + 127u) / 128u) * 128u;
}

static LaunchPlan plan_launch(const ks_sim* s) {
  LaunchPlan pl;
  pl.smem = (size_t)8 * (size_t)s->L;
  pl.decoupled = false; pl.rel_side = 0; pl.ring = 0; pl.group = 1; pl.mix = false; pl.rel_stride = 0; pl.mk_off = pl.mom_off = pl.mom_side = 0;
  int k = (int)(kSmemPerSM / ((long long)pl.smem + kSmemCtaOverhead));
  if (k < 1) k = 1;
  if (k > 32) k = 32;
  int T = 32;
  if (s->opt_threads) {
    T = s->opt_threads;
  } else {
    // few markets: widen until the grid brings ~16 warps to every SM (wider CTAs pay more at the
    // two barriers than their extra warps hide)
    const long long want_threads = (long long)s->num_sms * 512;
    const int a_cap = s->A > 32 ? s->A : 32;
    while (T < 1024 && (long long)s->M * T < want_threads && T * 2 <= a_cap) T *= 2;
    while (T < 1024 && (long long)k * T < 1024 && T * 2 <= a_cap) T *= 2;
  }
  pl.T = T;
  // ks_decoupled_kernel: legal for the zero-intelligence rules (literal or PACKED4) with plain
  // atomics when book + the ring of relative histograms fit the CTA's shared memory.  Automatic
  //  (a) when the grid leaves the GPU underfilled, i.e. the step latency is what counts (C1, C3):
  //      4k generating warps holding <= 3 events per thread + the clearing warp (T = 160/288/544),
  //      ring of 4;
  //  (b) when the SM holds only a few markets (C2: 6.9 per SM): there the persistent kernel's
  //      markets cannot hide each other's clearing, and 7 resident CTAs of 4 generating warps + 1
  //      clearing warp (T = 160) win.  Measured on B200, L = 256, delta = 16, A = 256..4096:
  //      the decoupled kernel is faster up to M = 2048 (13.8 markets per SM: +4 % .. +37 %) and
  //      slower at M = 4096 (-2 % .. -10 %), where the persistent kernel runs one warp per market.
  //  (d) the three-type population (KS_MODEL_MIX3, literal draws): two steps per pass with every rule
  //      relative to the step's opening price (generate_mix3_rel_group); needs >= 4 events per
  //      generating thread and class, small maker / momentum ranges (<= 64 bins) and four CTAs per SM.
  if (s->p.model == KS_MODEL_MIX3 && !s->opt_atomic && s->opt_pipe != 1 && s->opt_pair != 1 && !s->opt_cols && s->opt_ring == 0 &&
      s->p.maker_spread_max <= 64 && s->p.mom_delta + 1 <= 64) {
    const uint32_t side = rel_side_for(s);
    const uint32_t mk = (((uint32_t)s->p.maker_spread_max * 4u + 127u) / 128u) * 128u;
    const uint32_t ms = (((uint32_t)(s->p.mom_delta + 1) * 4u + 127u) / 128u) * 128u;
    const uint32_t stride = 2 * side + mk + 2 * ms;
    const size_t gsmem = pl.smem + 4 * (size_t)stride;
    const bool underfilled = (long long)s->M * pl.T < (long long)s->num_sms * 512;
    const bool legal = gsmem + 2048 <= (size_t)s->dev_smem_optin;
    const bool fit4 = 4 * ((long long)gsmem + kSmemCtaOverhead) <= kSmemPerSM;
    const bool autom = legal && fit4 && !underfilled && !s->opt_threads && s->A >= 3 * 128 * 4 && s->opt_pipe != 2;
    if (legal && (s->opt_pair == 2 || s->opt_pipe == 2 || (s->opt_pair == 0 && autom))) {
      const int Td = s->opt_threads ? s->opt_threads : 160;
      if (Td >= 64 && Td <= 160) {
        pl.T = Td; pl.decoupled = true; pl.rel_side = side; pl.ring = 4; pl.group = 2; pl.mix = true; pl.smem = gsmem;
        pl.rel_stride = stride; pl.mk_off = 2 * side; pl.mom_off = 2 * side + mk; pl.mom_side = ms;
        return pl;
      }
    }
  }
  const bool zi = s->p.model == KS_MODEL_ZI || s->p.model == KS_MODEL_ZI_PACKED4;
  if (zi && !s->opt_atomic && s->opt_pipe != 1) {
    const bool underfilled = (long long)s->M * pl.T < (long long)s->num_sms * 512;
    const bool few_per_sm = (long long)s->M <= 16LL * s->num_sms;
    const uint32_t side = rel_side_for(s);
    // ring depth: 4 histograms when the step latency counts, 2 when throughput does (half the code
    // in the instruction cache: C2 3.30 vs 3.38 ms); the lane-columned ablation layout has 2
    const int ring = s->opt_ring ? s->opt_ring : ((s->opt_cols || (long long)s->M > 2LL * s->num_sms) ? 2 : 4);
    const size_t dsmem = pl.smem + 2 * (size_t)ring * side;
    const bool fits = dsmem + 2048 <= (size_t)s->dev_smem_optin && !(s->opt_cols && ring != 2);
    const bool seven_fit = 7 * ((long long)dsmem + kSmemCtaOverhead) <= kSmemPerSM;
    // (c) two steps per pass (GROUP = 2, ring of 4, the clearing warp keeps the record): the literal
    //     contract with plain bins, >= 4 events per generating thread, seven CTAs fitting an SM, and
    //     the grid not underfilled.  Measured on B200 (L = 256 / 512): faster than every other plan
    //     for A >= 512 when an SM holds few markets (C2: 3.21 -> 2.99 ms) and for A >= 1024 at any M
    //     (C4: 640 ms persistent -> 608 ms with T = 96); slower for 2 events per thread (A = 256).
    const size_t gsmem = pl.smem + 8 * (size_t)side;
    const bool group_legal = s->p.model == KS_MODEL_ZI && !s->opt_cols && s->opt_ring == 0 && s->opt_pair != 1 &&
                             gsmem + 2048 <= (size_t)s->dev_smem_optin;
    const bool group_fit7 = 7 * ((long long)gsmem + kSmemCtaOverhead) <= kSmemPerSM;
    const bool group_auto = group_legal && group_fit7 && !underfilled && !s->opt_threads &&
                            ((few_per_sm && s->A >= 512) || s->A >= 1024);
    if (group_legal && (s->opt_pair == 2 || (s->opt_pair == 0 && group_auto))) {
      int Td = s->opt_threads ? s->opt_threads : (few_per_sm ? 160 : 96);
      if (Td >= 64 && Td <= 160) {
        pl.T = Td; pl.decoupled = true; pl.rel_side = side; pl.ring = 4; pl.group = 2; pl.smem = gsmem;
        return pl;
      }
    }
    if (fits && (s->opt_pipe == 2 || underfilled || (few_per_sm && seven_fit))) {
      int Td = pl.T;
      if (!s->opt_threads) {
        if (s->A < 128) {
          Td = 32 + 32 * ((s->A + 31) / 32 > 0 ? (s->A + 31) / 32 : 1);     // a handful of agents: no idle generating warps
        } else {
          // 4k generating warps (one, two, four per scheduler) + the clearing warp; <= 3 events per
          // thread when the step latency counts, one generating warp per scheduler otherwise
          Td = 160;
          if ((long long)s->M <= 2LL * s->num_sms) {
            while (Td < 544 && (long long)(Td - 32) * 3 < s->A) Td = 2 * (Td - 32) + 32;
            if (s->M > s->num_sms && Td > 288) Td = 288;
          }
        }
      }
      if (Td >= 64) { pl.T = Td; pl.decoupled = true; pl.rel_side = side; pl.ring = ring; pl.smem = dsmem; }
    }
  }
  return pl;
}

// cudaFuncSetAttribute is host work that used to precede every launch (1000 times in ks_run_stepwise).
// MaxDynamicSharedMemorySize is only an upper limit, so it is raised monotonically: one cache per
// kernel instantiation and device holding the largest value set so far (+1; 0 = never set).
struct SmemAttrCache { std::atomic<long long> set_plus1[64]; };

template <class K>
static cudaError_t ensure_smem_attr(K kern, SmemAttrCache& c, size_t smem) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const bool cached = dev >= 0 && dev < 64;
  if (cached && c.set_plus1[dev].load(std::memory_order_acquire) >= (long long)smem + 1) return cudaSuccess;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  if (e != cudaSuccess) return e;
  if (cached) {
    long long cur = c.set_plus1[dev].load(std::memory_order_relaxed);
    while (cur < (long long)smem + 1 && !c.set_plus1[dev].compare_exchange_weak(cur, (long long)smem + 1)) {}
  }
  return cudaSuccess;
}

template <int MODEL, int ATOM, bool PACKED>
static cudaError_t launch_persistent(const ks::KernelParams& P, int T, size_t smem, cudaStream_t st) {
  auto kern = ks::ks_persistent_kernel<MODEL, ATOM, PACKED>;
  static SmemAttrCache cache;
  cudaError_t e = ensure_smem_attr(kern, cache, smem);
  if (e != cudaSuccess) return e;
  kern<<<P.M, T, smem, st>>>(P);
  return cudaGetLastError();
}

template <bool PACKED, int COLS, int NB, int MAXT, int MINB, int GROUP = 1, bool MIX = false>
static cudaError_t launch_decoupled_as(const ks::KernelParams& P, int T, size_t smem, cudaStream_t st) {
  auto kern = ks::ks_decoupled_kernel<PACKED, COLS, NB, MAXT, MINB, GROUP, MIX>;
  static SmemAttrCache cache;
  cudaError_t e = ensure_smem_attr(kern, cache, smem);
  if (e != cudaSuccess) return e;
  kern<<<P.M, T, smem, st>>>(P);
  return cudaGetLastError();
}

#ifndef KS_GROUP_MAXT
#define KS_GROUP_MAXT 160      // launch bounds of the two-steps-per-pass instantiation: 7 CTAs of 160 threads per SM
#define KS_GROUP_MINB 7        // (56 registers)
#endif
// The decoupled kernel's instantiations: ring of 4 histograms (default) -- with the register budget
// of 7 resident CTAs of <= 160 threads when the block is that small (C2: 6.9 markets per SM must all
// be resident) -- or the two-deep ring (ablation; the only one with lane-columned bins).
template <bool PACKED>
static cudaError_t launch_decoupled(const ks::KernelParams& P, int T, size_t smem, int cols, int ring, int group, cudaStream_t st) {
  if (cols) return launch_decoupled_as<PACKED, 32, 2, 1024, 1>(P, T, smem, st);
  if constexpr (!PACKED) {
    if (group == 2 && T <= 160) return launch_decoupled_as<false, 1, 4, KS_GROUP_MAXT, KS_GROUP_MINB, 2>(P, T, smem, st);
  }
  if (ring == 2) return T <= 160 ? launch_decoupled_as<PACKED, 1, 2, 160, 7>(P, T, smem, st)
                                 : launch_decoupled_as<PACKED, 1, 2, 1024, 1>(P, T, smem, st);
  if (T <= 160) return launch_decoupled_as<PACKED, 1, 4, 160, 7>(P, T, smem, st);
  return launch_decoupled_as<PACKED, 1, 4, 1024, 1>(P, T, smem, st);
}

// Cluster launch: grid = M*C CTAs in clusters of C (cluster <-> market), 8*L/C bytes of shared
// memory per CTA.
template <int MODEL, bool PACKED>
static cudaError_t launch_cluster(const ks::KernelParams& P, int C, int T, cudaStream_t st) {
  auto kern = ks::ks_cluster_kernel<MODEL, PACKED>;
  const size_t smem = (size_t)8 * (size_t)(P.L / C);
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3((unsigned)P.M * (unsigned)C, 1, 1);
  cfg.blockDim = dim3((unsigned)T, 1, 1);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)C; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, P);
}

static ks_status run_impl(ks_sim* s, int64_t S, void* stream, const char* who, int32_t* d_trace = nullptr) {
  if (!s) { set_err("%s: NULL handle", who); return KS_ERR_INVALID_ARG; }
  if (S < 0) { set_err("%s: S < 0", who); return KS_ERR_INVALID_ARG; }
  {
    ks_status f = check_flags(s, who);
    if (f != KS_OK) return f;
  }
  if (S == 0) return KS_OK;
  DeviceGuard guard(s->device);
  // The depth bound of the last ks_write_books: taken from the host copy if the check has finished,
  // otherwise the kernel reads the device word itself (never a host-side wait).
  if (s->bound_pending) {
    const cudaError_t q = cudaEventQuery(s->bound_event);
    if (q == cudaSuccess) {
      s->bound_pending = 0;
      if (s->h_words[0] == 0xffffffffffffffffull) { set_err("%s: ks_write_books stored a negative depth", who); return KS_ERR_INVALID_ARG; }
      s->resting_bound = (int64_t)s->h_words[0];
    } else if (q != cudaErrorNotReady) {
      set_err("%s: %s", who, cudaGetErrorString(q)); return KS_ERR_CUDA;
    }
  }
  const long double total_steps = (long double)s->steps_done + (long double)S;
  const long double inflow = total_steps * (long double)s->inflow_per_step;
  const long double known_resting = s->bound_pending ? 0.0L : (long double)s->resting_bound;
  if (known_resting + inflow >= 2147483648.0L) { set_err("%s: per-side depth could reach 2^31", who); return KS_ERR_OVERFLOW; }
  // 8 steps of head-room: the decoupled kernel's 32-bit loop counters advance by up to 8 steps (ring
  // depth, or twice the steps per pass) and compare `s + stride < S`
  if (total_steps + 8.0L >= 4294967296.0L) { set_err("%s: the step counter would pass 2^32 - 8", who); return KS_ERR_OVERFLOW; }

  ks::KernelParams P;
  memset(&P, 0, sizeof(P));
  P.books = books_ptr(s);
  P.recs = recs_ptr(s);
  uint32_t k0 = (uint32_t)(s->seed & 0xffffffffu), k1 = (uint32_t)(s->seed >> 32);
  for (int r = 0; r < 10; ++r) { P.k0[r] = k0; P.k1[r] = k1; k0 += ks::kPhiloxW0; k1 += ks::kPhiloxW1; }
  P.M = s->M; P.L = s->L; P.A = s->A; P.market_base = s->market_base;
  P.noise_delta = s->p.noise_delta; P.noise_n = 2 * s->p.noise_delta + 1; P.noise_qmax = s->p.noise_qmax;
  P.noise_n4 = 4 * P.noise_n; P.q_addend = 1ull << 32;
  P.maker_spread_max = s->p.maker_spread_max; P.maker_qty = s->p.maker_qty;
  P.mom_n = s->p.mom_delta + 1; P.mom_qmax = s->p.mom_qmax;
  P.dmax = s->p.noise_delta;
  if (s->p.model == KS_MODEL_PAPER) {
    if (s->p.maker_spread_max > P.dmax) P.dmax = s->p.maker_spread_max;
    if (P.dmax < 1) P.dmax = 1;
    P.dmax += 1;                                       // round-half-up can add one tick
    P.paper_n_noise = s->n_noise; P.paper_n_mom = s->p.paper_n_mom; P.paper_pmkt_q16 = s->p.paper_pmkt_q16;
  } else if ((s->p.model & 1) == KS_MODEL_MIX3) {
    if (s->p.maker_spread_max > P.dmax) P.dmax = s->p.maker_spread_max;
    if (s->p.mom_delta > P.dmax) P.dmax = s->p.mom_delta;
  }
  P.fresh = s->fresh;
  P.force_generic = s->opt_clear;
  P.trace = reinterpret_cast<int2*>(d_trace);
  P.S = S;
  P.orders_per_step = (long long)s->A + s->n_maker;
  P.host_flags = s->d_flags;
  if (s->bound_pending) {
    P.depth_word = scratch_ptr(s);
    P.depth_limit = (unsigned long long)(2147483647.0L - inflow);   // inflow < 2^31 was checked above
  }

  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e;
  // the kernel reads the pending check's word on the device: order it after the check even when the
  // caller runs on another stream than ks_write_books did (asynchronous, no host wait)
  if (s->bound_pending) KS_CUDA(cudaStreamWaitEvent(st, s->bound_event, 0));
  const bool paper = s->p.model == KS_MODEL_PAPER;
  const bool mix = !paper && (s->p.model & 1) == KS_MODEL_MIX3;
  const bool packed = !paper && s->p.model >= KS_MODEL_ZI_PACKED4;
  int C = s->opt_cluster;
  if (C == 0) C = s->L > kMaxLPerCta ? s->L / kMaxLPerCta : 1;
  if (C > 1 && paper) { set_err("%s: the paper agent model has no cluster path", who); return KS_ERR_UNSUPPORTED; }
  if (C > 1) {
    // cluster path: the C*T threads of a cluster share the agents
    int T = s->opt_threads ? s->opt_threads : 256;
    while (!s->opt_threads && T > 32 && (long long)C * (T / 2) >= s->A) T /= 2;
    int log2C = 0;
    while ((1 << log2C) < C) ++log2C;
    P.log2C = log2C;
    if ((long long)s->M * C > 0x7fffffffLL) { set_err("%s: M * cluster size exceeds the grid limit", who); return KS_ERR_UNSUPPORTED; }
    if (!packed) e = mix ? launch_cluster<1, false>(P, C, T, st) : launch_cluster<0, false>(P, C, T, st);
    else         e = mix ? launch_cluster<1, true>(P, C, T, st) : launch_cluster<0, true>(P, C, T, st);
  } else {
    const LaunchPlan pl = plan_launch(s);
    P.rel_side = pl.rel_side; P.rel_stride = pl.mix ? pl.rel_stride : 2 * pl.rel_side;
    P.rel_mk_off = pl.mk_off; P.rel_mom_off = pl.mom_off; P.rel_mom_side = pl.mom_side;
    if (pl.decoupled && pl.mix) {
      e = launch_decoupled_as<false, 1, 4, KS_GROUP_MAXT, KS_GROUP_MINB, 2, true>(P, pl.T, pl.smem, st);
    } else if (pl.decoupled) {
      e = packed ? launch_decoupled<true>(P, pl.T, pl.smem, s->opt_cols, pl.ring, pl.group, st)
                 : launch_decoupled<false>(P, pl.T, pl.smem, s->opt_cols, pl.ring, pl.group, st);
    } else if (paper)
      e = launch_persistent<2, 0, false>(P, pl.T, pl.smem, st);
    else if (packed)
      e = mix ? launch_persistent<1, 0, true>(P, pl.T, pl.smem, st) : launch_persistent<0, 0, true>(P, pl.T, pl.smem, st);
    else if (!mix)
      e = s->opt_atomic ? launch_persistent<0, 1, false>(P, pl.T, pl.smem, st) : launch_persistent<0, 0, false>(P, pl.T, pl.smem, st);
    else
      e = s->opt_atomic ? launch_persistent<1, 1, false>(P, pl.T, pl.smem, st) : launch_persistent<1, 0, false>(P, pl.T, pl.smem, st);
  }
  if (e != cudaSuccess) { set_err("%s: launch failed: %s", who, cudaGetErrorString(e)); return KS_ERR_CUDA; }
  g_launches++;
  s->steps_done += S;
  s->fresh = 0;
  return KS_OK;
}

extern "C" {

ks_status ks_run(ks_sim* s, int64_t S, void* stream) { return run_impl(s, S, stream, "ks_run"); }

ks_status ks_run_traced(ks_sim* s, int64_t S, int32_t* d_trace, void* stream) {
  if (!d_trace) { set_err("ks_run_traced: NULL trace buffer"); return KS_ERR_INVALID_ARG; }
  if ((reinterpret_cast<uintptr_t>(d_trace) & 7) != 0) { set_err("ks_run_traced: d_trace must be 8-byte aligned"); return KS_ERR_INVALID_ARG; }
  return run_impl(s, S, stream, "ks_run_traced", d_trace);
}

ks_status ks_trace_stats(const int32_t* d_trace, int32_t M, int64_t S, int32_t K, double* d_out, void* stream) {
  if (!d_trace || !d_out || M < 1 || S < 1 || K < 0 || K > 256) { set_err("ks_trace_stats: bad argument"); return KS_ERR_INVALID_ARG; }
  const int warps = 4;
  ks::ks_trace_stats_kernel<<<(M + warps - 1) / warps, warps * 32, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<const int2*>(d_trace), M, (long long)S, K, d_out);
  KS_CUDA(cudaGetLastError());
  g_launches++;
  return KS_OK;
}

ks_status ks_plan_string(ks_sim* s, char* buf, size_t n) {
  if (!s || !buf || n == 0) { set_err("ks_plan_string: bad argument"); return KS_ERR_INVALID_ARG; }
  int C = s->opt_cluster;
  if (C == 0) C = s->L > kMaxLPerCta ? s->L / kMaxLPerCta : 1;
  if (C > 1) {
    snprintf(buf, n, "ks_cluster_kernel C=%d", C);
    return KS_OK;
  }
  const LaunchPlan pl = plan_launch(s);
  if (pl.decoupled)
    snprintf(buf, n, "ks_decoupled_kernel T=%d ring=%d steps_per_pass=%d%s%s", pl.T, pl.ring, pl.group, s->opt_cols ? " lane_columns" : "",
             pl.mix ? " mix3" : "");
  else
    snprintf(buf, n, "ks_persistent_kernel T=%d", pl.T);
  return KS_OK;
}

ks_status ks_error_state(ks_sim* s) {
  if (!s) { set_err("ks_error_state: NULL handle"); return KS_ERR_INVALID_ARG; }
  return check_flags(s, "ks_error_state");
}

ks_status ks_read_books(ks_sim* s, int32_t* dst, void* stream) {
  if (!s || !dst) { set_err("ks_read_books: NULL argument"); return KS_ERR_INVALID_ARG; }
  ks_status f = check_flags(s, "ks_read_books");
  if (f != KS_OK) return f;
  DeviceGuard guard(s->device);
  KS_CUDA(cudaMemcpyAsync(dst, books_ptr(s), (size_t)s->M * 8 * (size_t)s->L, cudaMemcpyDefault, (cudaStream_t)stream));
  return KS_OK;
}

ks_status ks_read_stats(ks_sim* s, ks_market_stats* dst, void* stream) {
  if (!s || !dst) { set_err("ks_read_stats: NULL argument"); return KS_ERR_INVALID_ARG; }
  ks_status f = check_flags(s, "ks_read_stats");
  if (f != KS_OK) return f;
  DeviceGuard guard(s->device);
  KS_CUDA(cudaMemcpyAsync(dst, recs_ptr(s), (size_t)s->M * 128, cudaMemcpyDefault, (cudaStream_t)stream));
  return KS_OK;
}

ks_status ks_write_books(ks_sim* s, const int32_t* src, void* stream) {
  if (!s || !src) { set_err("ks_write_books: NULL argument"); return KS_ERR_INVALID_ARG; }
  ks_status f = check_flags(s, "ks_write_books");
  if (f != KS_OK) return f;
  DeviceGuard guard(s->device);
  cudaStream_t st = (cudaStream_t)stream;
  KS_CUDA(cudaMemcpyAsync(books_ptr(s), src, (size_t)s->M * 8 * (size_t)s->L, cudaMemcpyDefault, st));
  s->fresh = 0;
  return enqueue_depth_check(s, st);
}

void ks_derive_stats(const ks_market_stats* rec, ks_derived_stats* out, int64_t n) {
  const double nan = std::nan("");
  for (int64_t i = 0; i < n; ++i) {
    const int64_t* f = rec[i].f;
    double* d = out[i].d;
    const double steps = (double)f[0], ntr = (double)f[1], vol = (double)f[2];
    d[0] = f[1] > 0 ? (double)f[3] / ntr : nan;
    d[1] = f[2] > 0 ? (double)f[5] / vol : nan;
    d[2] = f[0] > 0 ? vol / steps : nan;
    if (f[0] > 0) {
      const double mu = (double)f[6] / steps;
      const double var = (double)f[7] / steps - mu * mu;
      const double m4 = ((double)f[9] - 4.0 * mu * (double)f[8] + 6.0 * mu * mu * (double)f[7]) / steps -
                        3.0 * mu * mu * mu * mu;
      d[3] = mu; d[4] = var;
      d[5] = var > 0 ? m4 / (var * var) - 3.0 : nan;
    } else {
      d[3] = d[4] = d[5] = nan;
    }
  }
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------
// ks_depth_bound_static -- the depth check for callers who cannot allocate (include/kineticsim.h says
// who they are and why).  Every other kernel of this library works in memory the caller handed over;
// this one works in an array that is part of the library image itself, so the call needs neither a
// ks_sim nor a d_state and never asks the driver for memory.
//
// Layout of the array (8-byte words): [0] ticket counter, [1..31] unused (keeps the totals on their own
// 256-byte line), [32 + b] depth total of side b = 2*market + side.  It costs 1 MiB + 256 B of every
// GPU that loads the library, until the process exits.
//
// g_static_scratch below is two different things.  Inside device code the name IS the array.  In
// host code the same name is only a handle the runtime recognises -- it is not a device address, and a
// kernel (or cudaMemsetAsync) handed `g_static_scratch` from the host would touch some unrelated host
// location or fault.  The host therefore asks cudaGetSymbolAddress for the real address, once per
// device and with that device current (each GPU has its own copy at its own address), and passes that.
// ---------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned long long g_static_scratch[32 + 2 * KS_DEPTH_BOUND_STATIC_MAX_M];

namespace {

constexpr int kStaticMaxDevices = 64;
// device address of g_static_scratch per device ordinal; 0 = not looked up yet.  Two threads that
// race on the first call both store the same value.
std::atomic<unsigned long long*> g_static_addr[kStaticMaxDevices];

// One block per (market, side), as ks_depth_bound_kernel; instead of an atomicMax into a word of the
// caller's d_state, each block leaves its total in the library's array and takes a ticket, and the
// block that draws the last ticket reduces all totals into *out.
//   scratch[0] must be 0 at launch (the host clears it on the same stream); scratch[32 + b] is written
//   by block b before it is read by the last block, so stale totals of an earlier, larger call are
//   never looked at.
__global__ void ks_depth_bound_static_kernel(const int32_t* __restrict__ books, int L, unsigned long long* scratch,
                                             unsigned long long* out) {
  const int32_t* side = books + (size_t)blockIdx.x * (size_t)L;      // grid = 2*M sides
  long long sum = 0; int neg = 0;
  for (int i = threadIdx.x; i < L; i += blockDim.x) { const int v = side[i]; sum += v; neg |= (v < 0); }
  for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
  neg = __any_sync(0xffffffffu, neg);
  __shared__ long long s_sum[32];
  __shared__ int s_neg, s_last;
  if (threadIdx.x == 0) { s_neg = 0; s_last = 0; }
  __syncthreads();
  if ((threadIdx.x & 31) == 0) { s_sum[threadIdx.x >> 5] = sum; if (neg) s_neg = 1; }
  __syncthreads();
  if (threadIdx.x == 0) {
    long long tot = 0;
    for (int w = 0; w < (int)((blockDim.x + 31) >> 5); ++w) tot += s_sum[w];
    volatile unsigned long long* totals = scratch + 32;
    totals[blockIdx.x] = s_neg ? 0xffffffffffffffffull : (unsigned long long)tot;
    __threadfence();                                                 // total visible before the ticket
    const unsigned long long ticket = atomicAdd(&scratch[0], 1ull);
    s_last = ticket == (unsigned long long)gridDim.x - 1ull;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();                                                   // every other block's total is visible now
  const volatile unsigned long long* totals = scratch + 32;
  unsigned long long best = 0;
  for (unsigned b = threadIdx.x; b < gridDim.x; b += blockDim.x) { const unsigned long long v = totals[b]; best = v > best ? v : best; }
  for (int d = 16; d > 0; d >>= 1) { const unsigned long long o = __shfl_xor_sync(0xffffffffu, best, d); best = o > best ? o : best; }
  __shared__ unsigned long long s_best[32];
  if ((threadIdx.x & 31) == 0) s_best[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)((blockDim.x + 31) >> 5); ++w) best = s_best[w] > best ? s_best[w] : best;
    *out = best;
  }
}

// Device address of the library's array on the CURRENT device; looked up on the first call per device.
ks_status static_scratch_here(unsigned long long** out) {
  int dev = -1;
  KS_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) { set_err("ks_depth_bound_static: device ordinal beyond %s", "63"); return KS_ERR_UNSUPPORTED; }
  unsigned long long* ptr = g_static_addr[dev].load(std::memory_order_acquire);
  if (!ptr) {
    KS_CUDA(cudaGetSymbolAddress((void**)&ptr, g_static_scratch));
    if (!ptr) { set_err("ks_depth_bound_static: cudaGetSymbolAddress returned a NULL address"); return KS_ERR_CUDA; }
    g_static_addr[dev].store(ptr, std::memory_order_release);
  }
  *out = ptr;
  return KS_OK;
}

}  // namespace

extern "C" ks_status ks_depth_bound_static(const int32_t* d_books, int32_t M, int32_t L, uint64_t* d_out, void* stream) {
  if (!d_books || !d_out) { set_err("ks_depth_bound_static: NULL argument"); return KS_ERR_INVALID_ARG; }
  if ((reinterpret_cast<uintptr_t>(d_books) & 3) != 0 || (reinterpret_cast<uintptr_t>(d_out) & 7) != 0) {
    set_err("ks_depth_bound_static: d_books must be 4-byte and d_out 8-byte aligned"); return KS_ERR_INVALID_ARG;
  }
  if (!shape_ok(M, L)) { set_err("ks_depth_bound_static: need M >= 1 and L a power of two in 32..32768"); return KS_ERR_INVALID_ARG; }
  if (M > KS_DEPTH_BOUND_STATIC_MAX_M) {
    snprintf(g_err, sizeof(g_err),
             "ks_depth_bound_static: M = %d exceeds KS_DEPTH_BOUND_STATIC_MAX_M = %d (the library's built-in scratch holds one "
             "word per market side); check the image in slices of markets, or use ks_write_books / ks_attach on a d_state",
             (int)M, (int)KS_DEPTH_BOUND_STATIC_MAX_M);
    return KS_ERR_UNSUPPORTED;
  }
  unsigned long long* scratch = nullptr;
  const ks_status r = static_scratch_here(&scratch);
  if (r != KS_OK) return r;
  cudaStream_t st = (cudaStream_t)stream;
  KS_CUDA(cudaMemsetAsync(scratch, 0, sizeof(unsigned long long), st));            // the ticket counter starts at zero
  ks_depth_bound_static_kernel<<<2 * M, 128, 0, st>>>(d_books, L, scratch, reinterpret_cast<unsigned long long*>(d_out));
  KS_CUDA(cudaGetLastError());
  g_launches++;
  return KS_OK;
}
