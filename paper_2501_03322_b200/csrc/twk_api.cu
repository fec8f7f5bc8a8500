// twk_api.cu -- the C ABI of include/twk.h: argument validation, workspace, kernel launches.  No torch types.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "../../include/twk.h"
#include "twk_adaptive.cuh"
#include "twk_refine1.cuh"
#include "twk_stage1.cuh"

namespace {

constexpr int kAssumedSMs = 148;        // B200; workspace sizing only (twk_workspace_bytes needs no GPU)
// stage 2 keeps this iteration's new records in a shared-memory tile next to the arena (the tile column doubles as the
// scratch of the point solve); at the 4096-sample capacity of stage 3 the tile would cost the second resident CTA
constexpr bool kStage2Scr = true, kStage2Tile = true;
constexpr int kStage2Cap = 512;         // sample capacity of refinement stage 2
constexpr int kStage2CtasPerSM = 6;
constexpr int kStage3CtasPerSM = 2;
#ifndef TWK_S3_THREADS
#define TWK_S3_THREADS 128
#endif
constexpr int kStage3Threads = TWK_S3_THREADS;   // four warps share the O(n) passes of a stage-3 iteration (twk_adaptive.cuh)
constexpr int kFixedTile = 128;
constexpr size_t kCarrySlots = 1024;    // stage 2 -> stage 3 carry-over slots (120 KB each); beyond them stage 3 recomputes
constexpr size_t kDefaultHandoffSlots = size_t(1) << 19;   // 524,288 slots x 14,592 B = 7.6 GB

thread_local char g_cuda_msg[256] = "";

struct Plan {
  int cap2, cap3;       // 0 = stage absent
  int grid2, grid3;
  size_t arena_doubles;
};

Plan make_plan(const twk_options& o, int sms) {
  Plan P{};
  const int maxs = o.max_samples;
  P.cap2 = (maxs >= 2 * twk::kThreads) ? (maxs < kStage2Cap ? maxs : kStage2Cap) : 0;
  P.cap3 = (maxs > kStage2Cap) ? maxs : 0;
  P.grid2 = P.cap2 ? sms * kStage2CtasPerSM : 0;
  P.grid3 = P.cap3 ? sms * kStage3CtasPerSM : 0;
  const size_t a2 = (size_t)P.grid2 * P.cap2, a3 = (size_t)P.grid3 * P.cap3;
  P.arena_doubles = (a2 > a3 ? a2 : a3) * twk::kRecDoubles;
  return P;
}

size_t align256(size_t x) { return (x + 255) & ~size_t(255); }

size_t handoff_slots(const twk_options& o, size_t max_sources) {
  if (o.max_samples < 2 * twk::kThreads) return 0;   // no refinement stage
  const size_t want = o.handoff_slots < 0 ? kDefaultHandoffSlots : (size_t)o.handoff_slots;
  return want < max_sources ? want : max_sources;
}

struct Layout {
  size_t counters, list1, list1b, list2, seeds, handoff, carry, arena, total;
  size_t slots, carry_slots;
};
Layout make_layout(const twk_options& o, size_t max_sources, int sms) {
  const Plan P = make_plan(o, sms);
  Layout L{};
  size_t off = 0;
  L.slots = handoff_slots(o, max_sources);
  L.counters = off; off += 256;
  L.list1 = off;    off += align256(max_sources * 4);
  L.list1b = off;   off += align256(max_sources * 4);   // entries stage 1.5 leaves to stage 2
  L.list2 = off;    off += align256(max_sources * 4);
  L.seeds = off;    off += align256(max_sources * twk::kSeedDoubles * 8);
  L.handoff = off;  off += align256(L.slots * twk::kHandDoubles * 8);
  // (a context without hand-over slots is the lean one: no carry-over either)
  L.carry_slots = (P.cap2 && P.cap3 && L.slots) ? (kCarrySlots < max_sources ? kCarrySlots : max_sources) : 0;
  L.carry = off;    off += align256(L.carry_slots * twk::carry_doubles(P.cap2 ? P.cap2 : 1) * 8);
  L.arena = off;    off += align256(P.arena_doubles * 8);
  L.total = off;
  return L;
}

bool valid_options(const twk_options& o) {
  return o.max_samples >= twk::kThreads &&
         o.max_samples <= 4096 && (o.subtract_avg_tol == 0 || o.subtract_avg_tol == 1) && o.handoff_slots >= -1 && o.slope_gate >= 0.0 && o.slope_cos >= 0.0 && o.slope_cos <= 1.0 &&
         (o.point_source_test == 0 || o.point_source_test == 1) && (o.hidden_crossing_guard == 0 || o.hidden_crossing_guard == 1) &&
         (o.frame == 0 || o.frame == 1);
}

int cuda_fail(cudaError_t e) {
  snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error: %s", cudaGetErrorString(e));
  return TWK_ECUDA;
}
#define TWK_CUDA(x)                         \
  do {                                      \
    cudaError_t e_ = (x);                   \
    if (e_ != cudaSuccess) return cuda_fail(e_); \
  } while (0)

}  // namespace

// stage 1: persistent CTAs of 64 threads, kS1CtasPerSM per SM.  Measured on config 3 (B200) with several 64-thread
// teams per CTA kept in step by CTA-wide barriers: 1 x 6 CTAs/SM 36.5 ms, 2 x 3: 36.0, 3 x 2: 38.3, 4 x 1: 47.8,
// 6 x 1: 43.7 -- coupling the teams costs more than the shared instruction stream saves, so one team per CTA it is.
void launch_stage1(int sms, long long n_sources, twk::Stage1Args a, cudaStream_t stream) {
  {   // powers of the first iteration's interval width (twk::link_const on the host)
    const double dth = twk::kTwoPi / double(twk::kThreads), dth2 = dth * dth, dth3 = dth2 * dth;
    a.K1.dth2 = dth2;
    a.K1.c24 = dth3 * (1.0 / 24.0);
    a.K1.c12 = dth * (1.0 / 12.0);
    a.K1.c48 = dth3 * (1.0 / 48.0);
  }
  const size_t smem = twk::stage1_smem_bytes();   // below the 48 KB default limit: no opt-in needed
  static_assert(twk::stage1_smem_bytes() <= 48 * 1024, "stage-1 shared memory needs the opt-in attribute");
  const long long resident = (long long)sms * twk::kS1CtasPerSM;
  // group size: about 8 groups per resident CTA, so that the cursor can even out what the groups cost (a group of 64 is
  // 0.3 ms of one CTA, and a batch of two waves used to end with half of the CTAs waiting for the other half), but not
  // below 16 sources (per-group set-up: a DRAM round trip and three barriers) unless the batch is too small to give every
  // CTA 16.  Measured (stage 1, one group per CTA up to 64 -> this): 113,664 config-3 sources 0.78 -> 0.68 ms, Fig.5
  // resonant map 1.42 -> 1.31 ms, config 5 0.89 -> 0.78 ms, 400,000 sources 2.36 -> 2.29 ms; 4 groups per CTA gain a little
  // less, 2 nothing.
  long long group = (n_sources + 8 * resident - 1) / (8 * resident);
  {
    const long long g1 = (n_sources + resident - 1) / resident;   // one group per CTA
    long long lo = g1 < 16 ? g1 : 16;
    if (lo < 4) lo = 4;
    if (group < lo) group = lo;
  }
  group = group > twk::kS1Group ? twk::kS1Group : group;
  a.group = (int)group;
  long long groups = (n_sources + group - 1) / group;
  // a large batch ends in small groups: its last two waves of 64-source groups go out as groups of 16, so that the
  // resident CTAs finish within a quarter of a group's time of each other
  a.n_big = groups;
  a.tail_group = (int)group;
  a.interleave = 0;
  a.il_shift = 0;
  if (group == twk::kS1Group && groups > 8 * resident) {
    a.n_big = groups - 2 * resident;
    a.tail_group = 16;
    groups = a.n_big + (n_sources - a.n_big * group + 15) / 16;
  } else {
    // a batch of a few waves at most: a group is made of blocks of consecutive sources spread evenly over the batch (block b
    // of group g starts at source (g + b * groups) * B), so that a run of expensive neighbours is shared by many CTAs.
    // B = 4 (one full 32-byte sector per seed row and block) for groups of 16 sources or more, single sources below.
    // Measured (stage 1, contiguous groups -> these): config 2 0.256 -> 0.09 ms, Fig.5 resonant map 1.67 -> 1.42 ms, 64
    // light curves of config 3 0.71 -> 0.5 ms; a batch of many waves (config 4) does not care and keeps its contiguous
    // groups (and their coalesced seed rows).
    a.il_shift = group >= 16 ? 2 : 0;
    const long long B = 1ll << a.il_shift;
    group = (group + B - 1) / B * B;
    const long long blocks = (n_sources + B - 1) / B, per_group = group / B;
    groups = (blocks + per_group - 1) / per_group;
    a.group = (int)group;
    a.tail_group = (int)group;
    a.n_big = groups;
    a.interleave = 1;
  }
  const int grid = (int)(groups < resident ? groups : resident);
  if (a.guard && a.interleave) twk::stage1_kernel<true, true><<<grid, twk::kThreads, smem, stream>>>(a);
  else if (a.guard) twk::stage1_kernel<true, false><<<grid, twk::kThreads, smem, stream>>>(a);
  else if (a.interleave) twk::stage1_kernel<false, true><<<grid, twk::kThreads, smem, stream>>>(a);
  else twk::stage1_kernel<false, false><<<grid, twk::kThreads, smem, stream>>>(a);
}

constexpr int kHostChunksMax = 8;
// twk_magnify_host splits batches of at least kHostSplitMin sources into chunks of about kHostChunk (measured on config 3,
// 4,096,000 sources, pinned host buffers: see DESIGN.md section 6)
constexpr size_t kHostSplitMin = (size_t)1 << 21;
#ifndef TWK_HOST_CHUNK
#define TWK_HOST_CHUNK ((size_t)1 << 21)
#endif
constexpr size_t kHostChunk = TWK_HOST_CHUNK;

struct twk_ctx {
  twk_options opt;
  size_t max_sources;
  int sms;
  Plan plan;
  Layout lay;
  char* ws;
  // host staging for twk_magnify_host (allocated on first use)
  char* stage;
  size_t stage_bytes;
  // twk_magnify_host on a large batch: copy streams and events that overlap the transfers of one chunk with the kernels
  // of another (created on first use)
  cudaStream_t copy_in, copy_out;
  cudaEvent_t ev_in[kHostChunksMax], ev_done[kHostChunksMax], ev_first, ev_last;
  int last_launches;
  int timing;            // record CUDA events around every stage (twk_enable_stage_timing)
  cudaEvent_t ev[5];     // start, after stage 0, after stage 1, after stage 2, after stage 3
  int ev_used;           // number of events recorded by the last call
};

extern "C" {

void twk_default_options(twk_options* opt) {
  if (!opt) return;
  opt->max_samples = 4096;
  opt->subtract_avg_tol = 1;
  opt->handoff_slots = -1;
  opt->slope_gate = 1e-5;
  opt->slope_cos = 0.70710678118654752;
  opt->point_source_test = 0;
  opt->hidden_crossing_guard = 0;
  opt->frame = 0;
}

size_t twk_workspace_bytes(const twk_options* opt, size_t max_sources) {
  twk_options o;
  twk_default_options(&o);
  if (opt) o = *opt;
  if (!valid_options(o)) return 0;
  // the refinement stages' record arena scales with the SM count: the current device's when there is one (what
  // twk_create will allocate), a B200's 148 otherwise (host-side arithmetic, no GPU needed)
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      sms <= 0) {
    cudaGetLastError();
    sms = kAssumedSMs;
  }
  return make_layout(o, max_sources, sms).total;
}

int twk_create(twk_ctx** ctx, const twk_options* opt, size_t max_sources) {
  if (!ctx) return TWK_EINVAL;
  *ctx = nullptr;
  twk_options o;
  twk_default_options(&o);
  if (opt) o = *opt;
  if (!valid_options(o) || max_sources == 0 || max_sources > (size_t)0x7fffffff) return TWK_EINVAL;
  int dev = 0, sms = 0;
  TWK_CUDA(cudaGetDevice(&dev));
  TWK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  twk_ctx* c = new (std::nothrow) twk_ctx();
  if (!c) return TWK_ENOMEM;
  c->opt = o;
  c->max_sources = max_sources;
  c->sms = sms;
  c->plan = make_plan(o, sms);
  c->lay = make_layout(o, max_sources, sms);
  c->ws = nullptr;
  c->stage = nullptr;
  c->stage_bytes = 0;
  c->copy_in = c->copy_out = nullptr;
  c->ev_first = c->ev_last = nullptr;
  for (int i = 0; i < kHostChunksMax; ++i) c->ev_in[i] = c->ev_done[i] = nullptr;
  c->last_launches = 0;
  c->timing = 0;
  c->ev_used = 0;
  for (int i = 0; i < 5; ++i) c->ev[i] = nullptr;
  cudaError_t e = cudaMalloc((void**)&c->ws, c->lay.total);
  if (e != cudaSuccess) {
    delete c;
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? TWK_ENOMEM : cuda_fail(e);
  }
  // opt in to the large dynamic shared memory of stage 3 (a per-function attribute shared by all contexts, so
  // always the maximum the build supports)
  e = cudaFuncSetAttribute(twk::adaptive_kernel<false, false, false, kStage3Threads>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)twk::adaptive_smem_bytes(4096, false, false, kStage3Threads));
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(twk::adaptive_kernel<true, false, false, kStage3Threads>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)twk::adaptive_smem_bytes(4096, false, false, kStage3Threads));
  if (e != cudaSuccess) {
    cudaFree(c->ws);
    delete c;
    return cuda_fail(e);
  }
  *ctx = c;
  return TWK_OK;
}

int twk_destroy(twk_ctx* ctx) {
  if (!ctx) return TWK_OK;
  if (ctx->ws) cudaFree(ctx->ws);
  if (ctx->stage) cudaFree(ctx->stage);
  for (int i = 0; i < 5; ++i)
    if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
  for (int i = 0; i < kHostChunksMax; ++i) {
    if (ctx->ev_in[i]) cudaEventDestroy(ctx->ev_in[i]);
    if (ctx->ev_done[i]) cudaEventDestroy(ctx->ev_done[i]);
  }
  if (ctx->ev_first) cudaEventDestroy(ctx->ev_first);
  if (ctx->ev_last) cudaEventDestroy(ctx->ev_last);
  if (ctx->copy_in) cudaStreamDestroy(ctx->copy_in);
  if (ctx->copy_out) cudaStreamDestroy(ctx->copy_out);
  delete ctx;
  return TWK_OK;
}

static int check_batch(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                       size_t n_sources, const int32_t* model_id, const double* zeta) {
  if (!ctx) return TWK_EINVAL;
  if (n_sources == 0) return TWK_OK;
  if (!s || !q || !rho || !zeta || n_models == 0) return TWK_EINVAL;
  if (n_sources > ctx->max_sources) return TWK_EINVAL;
  if (!model_id && n_models != 1 && n_models != n_sources) return TWK_EINVAL;
  return TWK_OK;
}

static int magnify_impl(twk_ctx* ctx, const twk::Batch& batch, double rel_tol, double* out_mu, double* out_err,
                        int32_t* out_nsamples, uint32_t* out_status, void* stream_);

int twk_magnify(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho, size_t n_sources,
                const int32_t* model_id, const double* zeta, double rel_tol, double* out_mu, double* out_err,
                int32_t* out_nsamples, uint32_t* out_status, void* stream_) {
  const int rc = check_batch(ctx, n_models, s, q, rho, n_sources, model_id, zeta);
  if (rc != TWK_OK) return rc;
  if (n_sources == 0) return TWK_OK;
  if (!out_mu || !(rel_tol > 0.0)) return TWK_EINVAL;
  const twk::Batch b{s, q, rho, model_id, zeta, (long long)n_models, (long long)n_sources, ctx->opt.frame,
                     nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  return magnify_impl(ctx, b, rel_tol, out_mu, out_err, out_nsamples, out_status, stream_);
}

int twk_magnify_lightcurve(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                           const double* t0, const double* u0, const double* tE, const double* alpha, size_t n_sources,
                           const int32_t* model_id, const double* t, double rel_tol, double* out_mu, double* out_err,
                           int32_t* out_nsamples, uint32_t* out_status, void* stream_) {
  const int rc = check_batch(ctx, n_models, s, q, rho, n_sources, model_id, t);
  if (rc != TWK_OK) return rc;
  if (n_sources == 0) return TWK_OK;
  if (!t0 || !u0 || !tE || !alpha || !out_mu || !(rel_tol > 0.0)) return TWK_EINVAL;
  const twk::Batch b{s, q, rho, model_id, nullptr, (long long)n_models, (long long)n_sources, ctx->opt.frame,
                     t, t0, u0, tE, alpha, nullptr, nullptr};
  return magnify_impl(ctx, b, rel_tol, out_mu, out_err, out_nsamples, out_status, stream_);
}

int twk_magnify_lightcurve_orbital(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                                   const double* t0, const double* u0, const double* tE, const double* alpha,
                                   const double* ds_dt, const double* dalpha_dt, size_t n_sources, const int32_t* model_id,
                                   const double* t, double rel_tol, double* out_mu, double* out_err, int32_t* out_nsamples,
                                   uint32_t* out_status, void* stream_) {
  const int rc = check_batch(ctx, n_models, s, q, rho, n_sources, model_id, t);
  if (rc != TWK_OK) return rc;
  if (n_sources == 0) return TWK_OK;
  if (!t0 || !u0 || !tE || !alpha || !ds_dt || !dalpha_dt || !out_mu || !(rel_tol > 0.0)) return TWK_EINVAL;
  const twk::Batch b{s, q, rho, model_id, nullptr, (long long)n_models, (long long)n_sources, ctx->opt.frame,
                     t, t0, u0, tE, alpha, ds_dt, dalpha_dt};
  return magnify_impl(ctx, b, rel_tol, out_mu, out_err, out_nsamples, out_status, stream_);
}

static int magnify_impl(twk_ctx* ctx, const twk::Batch& batch, double rel_tol, double* out_mu, double* out_err,
                        int32_t* out_nsamples, uint32_t* out_status, void* stream_) {
  const size_t n_sources = (size_t)batch.n_sources;
  cudaStream_t stream = (cudaStream_t)stream_;
  const Plan& P = ctx->plan;
  int* counters = reinterpret_cast<int*>(ctx->ws + ctx->lay.counters);
  // counters: [0] cursor1, [1] count1 (refinement worklist), [2] cursor2, [3] count2 (stage-3 worklist), [4] cursor3,
  //           [5] cursor of stage 1.5, [6] count1b (entries stage 1.5 leaves to stage 2)
  TWK_CUDA(cudaMemsetAsync(counters, 0, 64, stream));
  twk::AdaptArgs a{};
  a.b = batch;
  a.tol = rel_tol;
  a.slope_gate2 = ctx->opt.slope_gate * ctx->opt.slope_gate;
  a.slope_cos2 = ctx->opt.slope_cos * ctx->opt.slope_cos;
  a.subtract_avg_tol = ctx->opt.subtract_avg_tol;
  a.guard = ctx->opt.hidden_crossing_guard;
  a.out_mu = out_mu;
  a.out_err = out_err;
  a.out_nsamples = out_nsamples;
  a.out_status = out_status;
  a.arena = reinterpret_cast<double*>(ctx->ws + ctx->lay.arena);
  double* handoff = reinterpret_cast<double*>(ctx->ws + ctx->lay.handoff);
  int32_t* list1 = reinterpret_cast<int32_t*>(ctx->ws + ctx->lay.list1);
  int32_t* list2 = reinterpret_cast<int32_t*>(ctx->ws + ctx->lay.list2);
  int launches = 0;
  ctx->ev_used = 0;
  auto mark = [&]() {
    if (ctx->timing && ctx->ev_used < 5) cudaEventRecord(ctx->ev[ctx->ev_used++], stream);
  };
  mark();
  // ---- stage 0: the point source at every source centre -> seed blocks --------------------------------------------
  double* seeds = reinterpret_cast<double*>(ctx->ws + ctx->lay.seeds);
  a.seeds = seeds;
  {
    const long long want = ((long long)n_sources + twk::kS0Threads - 1) / twk::kS0Threads;
    const long long cap = (long long)ctx->sms * 256;   // (a thread per source up to 4.8 M sources: the hardware balances the uneven solves best; measured 16 / 48 / 96 / 256 blocks per SM: 1.17 / 1.12 / 1.09 / 1.05 ms)
    twk::seeds_kernel<<<(int)(want < cap ? want : cap), twk::kS0Threads, 0, stream>>>(batch, seeds);
    ++launches;
  }
  mark();
  // ---- stage 1: every source, 64 samples, groups of 64 sources per CTA, everything in shared memory ----------------
  {
    twk::Stage1Args a1{};
    a1.b = a.b;
    a1.tol = rel_tol;
    a1.ps_test = ctx->opt.point_source_test;
    a1.guard = ctx->opt.hidden_crossing_guard;
    a1.slope_gate2 = ctx->opt.slope_gate * ctx->opt.slope_gate;
    a1.slope_cos2 = ctx->opt.slope_cos * ctx->opt.slope_cos;
    a1.final_stage = P.cap2 ? 0 : 1;
    a1.seeds = seeds;
    a1.cursor = counters + 0;
    a1.list = list1;
    a1.list_count = counters + 1;
    a1.handoff = handoff;
    a1.handoff_slots = (long long)ctx->lay.slots;
    a1.out_mu = out_mu;
    a1.out_err = out_err;
    a1.out_nsamples = out_nsamples;
    a1.out_status = out_status;
    launch_stage1(ctx->sms, (long long)n_sources, a1, stream);
    ++launches;
    mark();
  }
  // ---- stage 1.5: the first refinement iteration of the handed-over sources, all in shared memory (twk_refine1.cuh).
  //      Not with the L-4 guard (its term needs the neighbours' neighbours) and not without hand-over slots.
  const bool stage15 = P.cap2 >= 2 * twk::kThreads && ctx->lay.slots > 0 && !ctx->opt.hidden_crossing_guard;
  int32_t* list1b = reinterpret_cast<int32_t*>(ctx->ws + ctx->lay.list1b);
  if (stage15) {
    twk::Refine1Args r{};
    r.b = a.b;
    r.tol = rel_tol;
    r.slope_gate2 = a.slope_gate2;
    r.slope_cos2 = a.slope_cos2;
    r.subtract_avg_tol = a.subtract_avg_tol;
    r.list = list1;
    r.count = counters + 1;
    r.cursor = counters + 5;
    r.handoff = handoff;
    r.handoff_slots = (long long)ctx->lay.slots;
    r.next_list = list1b;
    r.next_count = counters + 6;
    r.out_mu = out_mu;
    r.out_err = out_err;
    r.out_nsamples = out_nsamples;
    r.out_status = out_status;
    twk::refine1_kernel<<<ctx->sms * kStage2CtasPerSM, twk::kThreads, twk::refine1_smem_bytes(), stream>>>(r);
    ++launches;
  }
  if (P.cap2) {
    // ---- stage 2: the worklist stage 1 appended (a9), first iteration handed over -------------------------------------
    twk::AdaptArgs a2 = a;
    a2.cap = P.cap2;
    a2.final_stage = P.cap3 ? 0 : 1;
    a2.list = list1;
    a2.count = stage15 ? counters + 6 : counters + 1;
    a2.remap = stage15 ? list1b : nullptr;
    a2.cursor = counters + 2;
    a2.next_list = list2;
    a2.next_count = counters + 3;
    a2.handoff = handoff;
    a2.handoff_slots = (long long)ctx->lay.slots;
    a2.carry = reinterpret_cast<double*>(ctx->ws + ctx->lay.carry);
    a2.carry_slots = (long long)ctx->lay.carry_slots;
    a2.carry_cap = P.cap2;
    a2.carry_role = (P.cap3 && ctx->lay.carry_slots) ? 1 : 0;
    constexpr bool kScr2 = kStage2Scr, kTile2 = kStage2Tile;
    const size_t smem2 = twk::adaptive_smem_bytes(P.cap2, kScr2, kTile2);
    if (a2.guard) twk::adaptive_kernel<true, kScr2, kTile2, twk::kThreads><<<P.grid2, twk::kThreads, smem2, stream>>>(a2);
    else twk::adaptive_kernel<false, kScr2, kTile2, twk::kThreads><<<P.grid2, twk::kThreads, smem2, stream>>>(a2);
    ++launches;
    mark();
  }
  if (P.cap3) {
    twk::AdaptArgs a3 = a;
    a3.cap = P.cap3;
    a3.final_stage = 1;
    a3.list = list2;
    a3.count = counters + 3;
    a3.cursor = counters + 4;
    a3.carry = reinterpret_cast<double*>(ctx->ws + ctx->lay.carry);
    a3.carry_slots = (long long)ctx->lay.carry_slots;
    a3.carry_cap = P.cap2;
    a3.carry_role = (P.cap2 && ctx->lay.carry_slots) ? 2 : 0;
    const size_t smem3 = twk::adaptive_smem_bytes(P.cap3, false, false, kStage3Threads);
    if (a3.guard) twk::adaptive_kernel<true, false, false, kStage3Threads><<<P.grid3, kStage3Threads, smem3, stream>>>(a3);
    else twk::adaptive_kernel<false, false, false, kStage3Threads><<<P.grid3, kStage3Threads, smem3, stream>>>(a3);
    ++launches;
    mark();
  }
  ctx->last_launches = launches;
  TWK_CUDA(cudaGetLastError());
  return TWK_OK;
}

static int images_fixed_impl(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                             size_t n_sources, const int32_t* model_id, const double* zeta, int N, double* out_z,
                             int8_t* out_kind, int8_t* out_count, double* out_mu, double* out_err, bool seeded,
                             uint32_t* out_diag, void* stream_) {
  const int rc = check_batch(ctx, n_models, s, q, rho, n_sources, model_id, zeta);
  if (rc != TWK_OK) return rc;
  if (n_sources == 0) return TWK_OK;
  if (N < 4) return TWK_EINVAL;
  cudaStream_t stream = (cudaStream_t)stream_;
  twk::Batch b{s, q, rho, model_id, zeta, (long long)n_models, (long long)n_sources, ctx->opt.frame,
               nullptr, nullptr, nullptr, nullptr, nullptr};
  const size_t smem = (size_t)(twk::kRecDoubles * kFixedTile + 2 * twk::kRecDoubles + 2 * (kFixedTile / 32) + 32) * 8;
  const long long resident = (long long)ctx->sms * 8;
  const int grid = (int)((long long)n_sources < resident ? (long long)n_sources : resident);
  if (seeded) {
    if (out_diag) TWK_CUDA(cudaMemsetAsync(out_diag, 0, 4 * sizeof(uint32_t), stream));
    twk::fixed_kernel<kFixedTile, true><<<grid, kFixedTile, smem, stream>>>(b, N, out_z, out_kind, out_count, out_mu, out_err, out_diag);
  } else {
    twk::fixed_kernel<kFixedTile, false><<<grid, kFixedTile, smem, stream>>>(b, N, out_z, out_kind, out_count, out_mu, out_err, nullptr);
  }
  ctx->last_launches = 1;
  TWK_CUDA(cudaGetLastError());
  return TWK_OK;
}

int twk_images_fixed(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                     size_t n_sources, const int32_t* model_id, const double* zeta, int N, double* out_z,
                     int8_t* out_kind, int8_t* out_count, double* out_mu, double* out_err, void* stream_) {
  return images_fixed_impl(ctx, n_models, s, q, rho, n_sources, model_id, zeta, N, out_z, out_kind, out_count, out_mu, out_err,
                           false, nullptr, stream_);
}

int twk_images_fixed_seeded(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                            size_t n_sources, const int32_t* model_id, const double* zeta, int N, double* out_z,
                            int8_t* out_kind, int8_t* out_count, double* out_mu, double* out_err, uint32_t* out_diag,
                            void* stream_) {
  return images_fixed_impl(ctx, n_models, s, q, rho, n_sources, model_id, zeta, N, out_z, out_kind, out_count, out_mu, out_err,
                           true, out_diag, stream_);
}

int twk_stage1_records(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho, size_t n_sources,
                       const int32_t* model_id, const double* zeta, double* out_records, uint32_t* out_diag, void* stream_) {
  const int rc = check_batch(ctx, n_models, s, q, rho, n_sources, model_id, zeta);
  if (rc != TWK_OK) return rc;
  if (n_sources == 0) return TWK_OK;
  if (!out_records) return TWK_EINVAL;
  cudaStream_t stream = (cudaStream_t)stream_;
  int* counters = reinterpret_cast<int*>(ctx->ws + ctx->lay.counters);
  TWK_CUDA(cudaMemsetAsync(counters, 0, 64, stream));
  if (out_diag) TWK_CUDA(cudaMemsetAsync(out_diag, 0, 4 * sizeof(uint32_t), stream));
  twk::Stage1Args a{};
  a.b = twk::Batch{s, q, rho, model_id, zeta, (long long)n_models, (long long)n_sources, ctx->opt.frame,
                   nullptr, nullptr, nullptr, nullptr, nullptr};
  {
    double* seeds = reinterpret_cast<double*>(ctx->ws + ctx->lay.seeds);
    const long long want = ((long long)n_sources + twk::kS0Threads - 1) / twk::kS0Threads;
    const long long cap = (long long)ctx->sms * 256;   // (a thread per source up to 4.8 M sources: the hardware balances the uneven solves best; measured 16 / 48 / 96 / 256 blocks per SM: 1.17 / 1.12 / 1.09 / 1.05 ms)
    twk::seeds_kernel<<<(int)(want < cap ? want : cap), twk::kS0Threads, 0, stream>>>(a.b, seeds);
    a.seeds = seeds;
  }
  a.tol = 1.0;                 // irrelevant: nothing is handed on (final_stage), nothing is written but the records
  a.slope_gate2 = ctx->opt.slope_gate * ctx->opt.slope_gate;
  a.slope_cos2 = ctx->opt.slope_cos * ctx->opt.slope_cos;
  a.ps_test = 0;
  a.final_stage = 1;
  a.cursor = counters + 0;
  a.list = reinterpret_cast<int32_t*>(ctx->ws + ctx->lay.list1);
  a.list_count = counters + 1;
  a.handoff = nullptr;
  a.handoff_slots = 0;
  a.dump = out_records;
  a.diag = out_diag;
  launch_stage1(ctx->sms, (long long)n_sources, a, stream);
  ctx->last_launches = 1;
  TWK_CUDA(cudaGetLastError());
  return TWK_OK;
}

int twk_coeffs_eq6(twk_ctx* ctx, size_t n_models, const double* s, const double* q, size_t n_sources, const int32_t* model_id,
                   const double* zeta, double* out_c, void* stream_) {
  const int rc = check_batch(ctx, n_models, s, q, s /* rho is not read */, n_sources, model_id, zeta);
  if (rc != TWK_OK) return rc;
  if (n_sources == 0) return TWK_OK;
  if (!out_c) return TWK_EINVAL;
  const twk::Batch b{s, q, s, model_id, zeta, (long long)n_models, (long long)n_sources, ctx->opt.frame};
  const long long want = ((long long)n_sources + 127) / 128;
  const int grid = (int)(want < (long long)ctx->sms * 16 ? want : (long long)ctx->sms * 16);
  twk::coeffs_kernel<<<grid, 128, 0, (cudaStream_t)stream_>>>(b, out_c);
  TWK_CUDA(cudaGetLastError());
  return TWK_OK;
}

int twk_magnify_host(twk_ctx* ctx, size_t n_models, const double* s, const double* q, const double* rho,
                     size_t n_sources, const int32_t* model_id, const double* zeta, double rel_tol, double* out_mu,
                     double* out_err, int32_t* out_nsamples, uint32_t* out_status, void* stream_) {
  const int rc = check_batch(ctx, n_models, s, q, rho, n_sources, model_id, zeta);
  if (rc != TWK_OK) return rc;
  if (n_sources == 0) return TWK_OK;
  if (!out_mu || !(rel_tol > 0.0)) return TWK_EINVAL;
  cudaStream_t stream = (cudaStream_t)stream_;
  // staging layout (device): s, q, rho [n_models each] | model_id | zeta | mu | err | nsamples | status
  const size_t need = align256(n_models * 8) * 3 + align256(n_sources * 4) + align256(n_sources * 16) +
                      align256(n_sources * 8) * 2 + align256(n_sources * 4) * 2;
  if (need > ctx->stage_bytes) {
    // (re)allocation happens on the first call and when a batch outgrows the staging area, which then at least doubles:
    // a sequence of calls of any sizes allocates O(log) times, none in the steady state
    if (ctx->stage) cudaFree(ctx->stage);
    ctx->stage = nullptr;
    const size_t grown = 2 * ctx->stage_bytes;
    ctx->stage_bytes = 0;
    const size_t want = need > grown ? need : grown;
    cudaError_t e = cudaMalloc((void**)&ctx->stage, want);
    if (e != cudaSuccess && want > need) {
      cudaGetLastError();
      e = cudaMalloc((void**)&ctx->stage, need);
      if (e == cudaSuccess) ctx->stage_bytes = need;
    } else if (e == cudaSuccess) {
      ctx->stage_bytes = want;
    }
    if (e != cudaSuccess) {
      cudaGetLastError();
      return e == cudaErrorMemoryAllocation ? TWK_ENOMEM : cuda_fail(e);
    }
  }
  char* p = ctx->stage;
  double* d_s = (double*)p;      p += align256(n_models * 8);
  double* d_q = (double*)p;      p += align256(n_models * 8);
  double* d_rho = (double*)p;    p += align256(n_models * 8);
  int32_t* d_mid = (int32_t*)p;  p += align256(n_sources * 4);
  double* d_zeta = (double*)p;   p += align256(n_sources * 16);
  double* d_mu = (double*)p;     p += align256(n_sources * 8);
  double* d_err = (double*)p;    p += align256(n_sources * 8);
  int32_t* d_ns = (int32_t*)p;   p += align256(n_sources * 4);
  uint32_t* d_st = (uint32_t*)p;
  TWK_CUDA(cudaMemcpyAsync(d_s, s, n_models * 8, cudaMemcpyHostToDevice, stream));
  TWK_CUDA(cudaMemcpyAsync(d_q, q, n_models * 8, cudaMemcpyHostToDevice, stream));
  TWK_CUDA(cudaMemcpyAsync(d_rho, rho, n_models * 8, cudaMemcpyHostToDevice, stream));
  if (n_sources < kHostSplitMin) {   // one piece, everything in stream order
    if (model_id) TWK_CUDA(cudaMemcpyAsync(d_mid, model_id, n_sources * 4, cudaMemcpyHostToDevice, stream));
    TWK_CUDA(cudaMemcpyAsync(d_zeta, zeta, n_sources * 16, cudaMemcpyHostToDevice, stream));
    const int r2 = twk_magnify(ctx, n_models, d_s, d_q, d_rho, n_sources, model_id ? d_mid : nullptr, d_zeta, rel_tol, d_mu,
                               out_err ? d_err : nullptr, out_nsamples ? d_ns : nullptr, out_status ? d_st : nullptr, stream_);
    if (r2 != TWK_OK) return r2;
    TWK_CUDA(cudaMemcpyAsync(out_mu, d_mu, n_sources * 8, cudaMemcpyDeviceToHost, stream));
    if (out_err) TWK_CUDA(cudaMemcpyAsync(out_err, d_err, n_sources * 8, cudaMemcpyDeviceToHost, stream));
    if (out_nsamples) TWK_CUDA(cudaMemcpyAsync(out_nsamples, d_ns, n_sources * 4, cudaMemcpyDeviceToHost, stream));
    if (out_status) TWK_CUDA(cudaMemcpyAsync(out_status, d_st, n_sources * 4, cudaMemcpyDeviceToHost, stream));
    TWK_CUDA(cudaStreamSynchronize(stream));
    return TWK_OK;
  }
  // A large batch goes through in chunks: the sources are independent, so the host->device copy of chunk c + 1 and
  // the device->host copy of chunk c - 1 run on two copy streams while the kernels of chunk c run on `stream`.  The chunks
  // share the context's workspace and are serialised on `stream`; only the transfers overlap.
  if (!ctx->copy_in) {
    TWK_CUDA(cudaStreamCreateWithFlags(&ctx->copy_in, cudaStreamNonBlocking));
    TWK_CUDA(cudaStreamCreateWithFlags(&ctx->copy_out, cudaStreamNonBlocking));
    TWK_CUDA(cudaEventCreateWithFlags(&ctx->ev_first, cudaEventDisableTiming));
    TWK_CUDA(cudaEventCreateWithFlags(&ctx->ev_last, cudaEventDisableTiming));
    for (int i = 0; i < kHostChunksMax; ++i) {
      TWK_CUDA(cudaEventCreateWithFlags(&ctx->ev_in[i], cudaEventDisableTiming));
      TWK_CUDA(cudaEventCreateWithFlags(&ctx->ev_done[i], cudaEventDisableTiming));
    }
  }
  // chunk boundaries: chunks of `per` sources, except that the first one is half that size -- its host->device copy and
  // the last chunk's device->host copy are the transfers nothing overlaps
  size_t per = kHostChunk, lim = (n_sources + kHostChunksMax - 2) / (kHostChunksMax - 1);
  if (per < lim) per = lim;
  per = (per + 8191) / 8192 * 8192;
  size_t bound[kHostChunksMax + 1];
  int n_chunks = 0;
  bound[0] = 0;
  for (size_t off = 0; off < n_sources;) {
    const size_t want = (n_chunks == 0) ? per / 2 : per;
    off = (n_sources - off <= want || n_chunks == kHostChunksMax - 1) ? n_sources : off + want;
    bound[++n_chunks] = off;
  }
  const bool identity = !model_id && n_models == n_sources && n_models > 1;   // model i belongs to source i
  // the copy streams start after what `stream` has been given so far (the parameters above; earlier calls that use
  // the staging area)
  TWK_CUDA(cudaEventRecord(ctx->ev_first, stream));
  TWK_CUDA(cudaStreamWaitEvent(ctx->copy_in, ctx->ev_first, 0));
  TWK_CUDA(cudaStreamWaitEvent(ctx->copy_out, ctx->ev_first, 0));
  for (int c = 0; c < n_chunks; ++c) {
    const size_t off = bound[c], m = bound[c + 1] - off;
    if (model_id) TWK_CUDA(cudaMemcpyAsync(d_mid + off, model_id + off, m * 4, cudaMemcpyHostToDevice, ctx->copy_in));
    TWK_CUDA(cudaMemcpyAsync(d_zeta + 2 * off, zeta + 2 * off, m * 16, cudaMemcpyHostToDevice, ctx->copy_in));
    TWK_CUDA(cudaEventRecord(ctx->ev_in[c], ctx->copy_in));
  }
  int launches = 0;
  for (int c = 0; c < n_chunks; ++c) {
    const size_t off = bound[c], m = bound[c + 1] - off;
    const size_t po = identity ? off : 0;
    TWK_CUDA(cudaStreamWaitEvent(stream, ctx->ev_in[c], 0));
    const int r2 = twk_magnify(ctx, identity ? m : n_models, d_s + po, d_q + po, d_rho + po, m, model_id ? d_mid + off : nullptr,
                               d_zeta + 2 * off, rel_tol, d_mu + off, out_err ? d_err + off : nullptr,
                               out_nsamples ? d_ns + off : nullptr, out_status ? d_st + off : nullptr, stream_);
    if (r2 != TWK_OK) {
      cudaStreamSynchronize(ctx->copy_in);
      cudaStreamSynchronize(ctx->copy_out);
      cudaStreamSynchronize(stream);
      return r2;
    }
    launches += ctx->last_launches;
    TWK_CUDA(cudaEventRecord(ctx->ev_done[c], stream));
    TWK_CUDA(cudaStreamWaitEvent(ctx->copy_out, ctx->ev_done[c], 0));
    TWK_CUDA(cudaMemcpyAsync(out_mu + off, d_mu + off, m * 8, cudaMemcpyDeviceToHost, ctx->copy_out));
    if (out_err) TWK_CUDA(cudaMemcpyAsync(out_err + off, d_err + off, m * 8, cudaMemcpyDeviceToHost, ctx->copy_out));
    if (out_nsamples) TWK_CUDA(cudaMemcpyAsync(out_nsamples + off, d_ns + off, m * 4, cudaMemcpyDeviceToHost, ctx->copy_out));
    if (out_status) TWK_CUDA(cudaMemcpyAsync(out_status + off, d_st + off, m * 4, cudaMemcpyDeviceToHost, ctx->copy_out));
  }
  ctx->last_launches = launches;
  TWK_CUDA(cudaEventRecord(ctx->ev_last, ctx->copy_out));
  TWK_CUDA(cudaStreamWaitEvent(stream, ctx->ev_last, 0));   // `stream` stays the one order of everything this call did
  TWK_CUDA(cudaStreamSynchronize(stream));
  return TWK_OK;
}

int twk_last_stats(twk_ctx* ctx, int64_t* n_stage2, int64_t* n_stage3, int* n_launches, void* stream_) {
  if (!ctx) return TWK_EINVAL;
  int h[8] = {0};
  TWK_CUDA(cudaMemcpyAsync(h, ctx->ws + ctx->lay.counters, sizeof(h), cudaMemcpyDeviceToHost, (cudaStream_t)stream_));
  TWK_CUDA(cudaStreamSynchronize((cudaStream_t)stream_));
  if (n_stage2) *n_stage2 = h[1];
  if (n_stage3) *n_stage3 = h[3];
  if (n_launches) *n_launches = ctx->last_launches;
  return TWK_OK;
}

int twk_enable_stage_timing(twk_ctx* ctx, int on) {
  if (!ctx) return TWK_EINVAL;
  if (on)
    for (int i = 0; i < 5; ++i)
      if (!ctx->ev[i]) TWK_CUDA(cudaEventCreate(&ctx->ev[i]));
  ctx->timing = on ? 1 : 0;
  ctx->ev_used = 0;
  return TWK_OK;
}

int twk_last_stage_ms(twk_ctx* ctx, float* ms4) {
  if (!ctx || !ms4) return TWK_EINVAL;
  for (int i = 0; i < 4; ++i) ms4[i] = 0.0f;
  if (!ctx->timing || ctx->ev_used < 2) return TWK_EINVAL;
  TWK_CUDA(cudaEventSynchronize(ctx->ev[ctx->ev_used - 1]));
  for (int i = 0; i + 1 < ctx->ev_used && i < 4; ++i) TWK_CUDA(cudaEventElapsedTime(&ms4[i], ctx->ev[i], ctx->ev[i + 1]));
  return TWK_OK;
}

int twk_fp64_peak_probe(int iters, double* out_tflops) {
  if (iters <= 0 || !out_tflops) return TWK_EINVAL;
  int dev = 0, sms = 0;
  TWK_CUDA(cudaGetDevice(&dev));
  TWK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double* d = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaStream_t st = nullptr;
  float best = 1e30f;
  const int grid = sms * 8, block = 256;
  cudaError_t err = cudaMalloc((void**)&d, 8);
  if (err == cudaSuccess) err = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking);
  if (err == cudaSuccess) err = cudaEventCreate(&e0);
  if (err == cudaSuccess) err = cudaEventCreate(&e1);
  if (err == cudaSuccess) {
    twk::dfma_probe_kernel<<<grid, block, 0, st>>>(iters / 8 + 1, d);   // warm-up
    for (int rep = 0; rep < 3 && err == cudaSuccess; ++rep) {
      cudaEventRecord(e0, st);
      twk::dfma_probe_kernel<<<grid, block, 0, st>>>(iters, d);
      cudaEventRecord(e1, st);
      err = cudaEventSynchronize(e1);
      float ms = 0;
      if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
      if (err == cudaSuccess && ms < best) best = ms;
    }
    if (err == cudaSuccess) err = cudaGetLastError();
  }
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  if (st) cudaStreamDestroy(st);
  if (d) cudaFree(d);
  if (err != cudaSuccess) {
    cudaGetLastError();
    return cuda_fail(err);
  }
  const double flop = 2.0 * 8.0 * (double)iters * (double)grid * (double)block;
  *out_tflops = flop / ((double)best * 1e-3) / 1e12;
  return TWK_OK;
}

// ---- twk_magnify_static: the adaptive path with NO allocation ------------------------------------------------------
// For callers that cannot call cudaMalloc (code under CUDA graph capture, serving loops, harnesses that forbid it): the
// workspace of the same kernels -- counters, worklists, seed blocks, the refinement stages' record arena -- lives in a
// file-scope __device__ array instead of a context's cudaMalloc'ed block.  Every GPU that loads the library holds the
// array (TWK_STATIC_SCRATCH_BYTES) until the process exits; every call on a device shares it.
namespace {
constexpr size_t kStaticMaxSources = TWK_STATIC_MAX_SOURCES;
constexpr int kStaticGrid2 = 128, kStaticGrid3 = 16;   // CTAs of the two refinement stages (each owns a slice of the arena)
constexpr int kStaticMaxDevices = 64;
constexpr size_t static_align256(size_t x) { return (x + 255) & ~size_t(255); }
constexpr size_t kStaticArenaRecords =
    (size_t)kStaticGrid2 * kStage2Cap > (size_t)kStaticGrid3 * 4096 ? (size_t)kStaticGrid2 * kStage2Cap : (size_t)kStaticGrid3 * 4096;
// counters | list1 | list1b | list2 | seed blocks | record arena (no hand-over and no carry-over slots: the lean layout)
constexpr size_t kStaticNeed = 256 + 3 * static_align256(kStaticMaxSources * 4) +
                               static_align256(kStaticMaxSources * twk::kSeedDoubles * 8) +
                               static_align256(kStaticArenaRecords * twk::kRecDoubles * 8);
static_assert(kStaticNeed <= TWK_STATIC_SCRATCH_BYTES, "TWK_STATIC_SCRATCH_BYTES too small for TWK_STATIC_MAX_SOURCES");
}  // namespace

// In host code this name is only a handle for cudaGetSymbolAddress: it is NOT a device address.
static __device__ __align__(256) unsigned char g_twk_static_scratch[TWK_STATIC_SCRATCH_BYTES];

namespace {
struct StaticSlot {
  bool ready;
  twk_ctx ctx;
};
StaticSlot g_static[kStaticMaxDevices];   // one per device, host memory of the library image (no allocation)
std::mutex g_static_mutex;

// Set-up, once per device, with that device current: the array's device address, the plan and the layout.
int static_context(twk_ctx** out) {
  int dev = 0;
  TWK_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) return TWK_EINVAL;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticSlot& S = g_static[dev];
  if (!S.ready) {
    int sms = 0;
    TWK_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    void* base = nullptr;
    TWK_CUDA(cudaGetSymbolAddress(&base, g_twk_static_scratch));
    if (!base) return TWK_ECUDA;
    twk_ctx& c = S.ctx;
    twk_default_options(&c.opt);
    c.opt.handoff_slots = 0;
    c.max_sources = kStaticMaxSources;
    c.sms = sms;
    c.plan = make_plan(c.opt, sms);
    c.plan.grid2 = kStaticGrid2;   // any grid works: the CTAs are persistent and fetch their sources from a cursor
    c.plan.grid3 = kStaticGrid3;
    c.plan.arena_doubles = kStaticArenaRecords * twk::kRecDoubles;
    Layout L{};
    size_t off = 0;
    L.counters = off; off += 256;
    L.list1 = off;    off += align256(kStaticMaxSources * 4);
    L.list1b = off;   off += align256(kStaticMaxSources * 4);
    L.list2 = off;    off += align256(kStaticMaxSources * 4);
    L.seeds = off;    off += align256(kStaticMaxSources * twk::kSeedDoubles * 8);
    L.handoff = off;
    L.carry = off;
    L.arena = off;    off += align256(c.plan.arena_doubles * 8);
    L.total = off;
    L.slots = 0;
    L.carry_slots = 0;
    if (L.total > sizeof(g_twk_static_scratch)) return TWK_EINVAL;   // (the static_assert above says it cannot be)
    c.lay = L;
    c.ws = static_cast<char*>(base);
    c.stage = nullptr;
    c.stage_bytes = 0;
    c.copy_in = c.copy_out = nullptr;
    c.ev_first = c.ev_last = nullptr;
    for (int i = 0; i < kHostChunksMax; ++i) c.ev_in[i] = c.ev_done[i] = nullptr;
    c.last_launches = 0;
    c.timing = 0;
    c.ev_used = 0;
    for (int i = 0; i < 5; ++i) c.ev[i] = nullptr;
    // the large dynamic shared memory of the last stage is a per-device function attribute (no allocation)
    TWK_CUDA(cudaFuncSetAttribute(twk::adaptive_kernel<false, false, false, kStage3Threads>,
                                  cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)twk::adaptive_smem_bytes(4096, false, false, kStage3Threads)));
    S.ready = true;
  }
  *out = &S.ctx;
  return TWK_OK;
}
}  // namespace

int twk_magnify_static(size_t n_models, const double* s, const double* q, const double* rho, size_t n_sources,
                       const int32_t* model_id, const double* zeta, double rel_tol, double* out_mu, double* out_err,
                       int32_t* out_nsamples, uint32_t* out_status, void* stream_) {
  if (n_sources > kStaticMaxSources) return TWK_ELIMIT;
  if (n_sources == 0) return TWK_OK;
  twk_ctx* ctx = nullptr;
  const int r0 = static_context(&ctx);
  if (r0 != TWK_OK) return r0;
  const int rc = check_batch(ctx, n_models, s, q, rho, n_sources, model_id, zeta);
  if (rc != TWK_OK) return rc;
  if (!out_mu || !(rel_tol > 0.0)) return TWK_EINVAL;
  const twk::Batch b{s, q, rho, model_id, zeta, (long long)n_models, (long long)n_sources, ctx->opt.frame,
                     nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  // (the call clears the 64 bytes of counters on the stream; every other part of the scratch is written before it is read)
  return magnify_impl(ctx, b, rel_tol, out_mu, out_err, out_nsamples, out_status, stream_);
}

int twk_debug_counters(uint32_t* out12, int reset) {
#ifdef TWK_DEBUG
  if (!out12) return TWK_EINVAL;
  TWK_CUDA(cudaDeviceSynchronize());
  TWK_CUDA(cudaMemcpyFromSymbol(out12, twk::g_twk_debug, 12 * sizeof(uint32_t)));
  if (reset) {
    uint32_t z[12] = {0};
    TWK_CUDA(cudaMemcpyToSymbol(twk::g_twk_debug, z, sizeof(z)));
  }
  return TWK_OK;
#else
  (void)out12;
  (void)reset;
  return TWK_EINVAL;   // not a debug build
#endif
}

const char* twk_strerror(int code) {
  switch (code) {
    case TWK_OK: return "ok";
    case TWK_EINVAL: return "invalid argument";
    case TWK_ENOMEM: return "out of device memory for the workspace";
    case TWK_ECUDA: return g_cuda_msg[0] ? g_cuda_msg : "CUDA runtime error";
    case TWK_ELIMIT: return "batch larger than TWK_STATIC_MAX_SOURCES, the limit of twk_magnify_static's fixed scratch (use a context)";
    default: return "unknown twk error code";
  }
}

#ifndef TWK_SOURCE_HASH
#define TWK_SOURCE_HASH "unknown"
#endif
#ifdef TWK_DEBUG
const char* twk_version(void) { return "twk 0.2 (sm_100a, TWK_DEBUG) src:" TWK_SOURCE_HASH; }
#else
const char* twk_version(void) { return "twk 0.2 (sm_100a) src:" TWK_SOURCE_HASH; }
#endif

}  // extern "C"
