// twk_kernels.cuh -- the kernels of the hot path (rows a8, a9 of SURVEY.md section 8(a) on top of the device
// functions a1-a7 in twk_device.cuh / twk_contour.cuh).
//
//   fixed_kernel      fixed-sampling mode: theta_j = 2 pi j / N, one CTA per source, records staged in shared memory
//   adaptive_kernel   the adaptive loop of P:318-326 for one source per CTA (64 or 128 threads), entirely on-device:
//                     64 samples per iteration (one thread each), per-source sorted sample state in shared memory,
//                     error-weighted inverse-transform sampling, stop rule + cap.
//                     Refinement stages 2/3 (twk_adaptive.cuh): records in a per-CTA global arena (L2 resident),
//                     sources taken from the worklist of the previous stage.  Stage 1 (twk_stage1.cuh) is the
//                     first iteration of every source, everything in shared memory.
//   refine1_kernel    stage 1.5 (twk_refine1.cuh): the first refinement iteration (64 -> up to 128 samples) of the sources
//                     stage 1 handed over, old and new records in two shared-memory tiles; what it cannot finish is left
//                     to stage 2 untouched.
//   coeffs_kernel     parity harness: the Eq.(6) coefficients as the device builds them
//   dfma_probe_kernel FP64 FMA throughput probe (roofline denominator)
#pragma once

#include <cuda_runtime.h>

#include "twk_contour.cuh"

namespace twk {

// ------------------------------------------------------------------------------------------------------------
// Debug build (-DTWK_DEBUG, libtwk_debug.so): the builder's own invariants, counted instead of trapped so that a
// violated one does not take the context down.  compute-sanitizer is not available on this pool; these checks are what
// stands in for memcheck / racecheck on the data-dependent indexing of the refinement kernels (tests/test_gpu_debug.py).
//   [0] record id outside the CTA's arena            [1] sample angles not strictly increasing after an iteration
//   [2] sorted list is not a permutation of the ids  [3] a record re-judged by two threads in one phase
//   [4] worklist / hand-over slot out of range       [5] a new angle outside the interval that owns its quantile
//   [6] sources checked by the refinement stages     [7] iterations checked
// and four plain event counts of stage 1.5 (twk_refine1.cuh):
//   [8] entries taken up                              [9] of those, entries whose new samples were solved
//   [10] of those, sources finished there             [11] entries passed on unread (no hand-over slot / stage 1's mark)
// ------------------------------------------------------------------------------------------------------------
#ifdef TWK_DEBUG
__device__ unsigned g_twk_debug[12];
__device__ unsigned g_twk_stamp[2048 * 64];   // one bit per record of every CTA's arena slot (<= 2048 CTAs x 4096 records)
#define TWK_CHECK(cond, which)                            \
  do {                                                    \
    if (!(cond)) atomicAdd(&twk::g_twk_debug[which], 1u); \
  } while (0)
#define TWK_DEBUG_COUNT(which) atomicAdd(&twk::g_twk_debug[which], 1u)
#else
#define TWK_CHECK(cond, which) \
  do {                         \
  } while (0)
#define TWK_DEBUG_COUNT(which) \
  do {                         \
  } while (0)
#endif

constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr double kPi = 3.141592653589793238462643383279;
constexpr double kInvPi = 0.318309886183790671537767526745;
constexpr int kThreads = 64;   // threads per source = samples per iteration
// Hand-over slot (stage 1 -> stage 2), in doubles: records [26][64] | dA [64] | err [64] | seed block [31] (+1 pad) |
// header [16]: source id (raw bits), s, m1, m2, z2, Re zc, Im zc, rho, status (raw bits) -- with the header the refinement
// stage needs ONE round trip to memory to start a handed-over source (no worklist / model / parameter chain)
constexpr int kHandHeader = (kRecDoubles + 2) * kThreads + 32;
constexpr int kHandDoubles = kHandHeader + 16;

struct Batch {
  const double* s;
  const double* q;
  const double* rho;
  const int32_t* model_id;   // may be null
  const double* zeta;        // [n][2]
  long long n_models, n_sources;
  int frame;                 // 0: zeta in the centre-of-mass frame (Eq.2); 1: primary at the origin (zeta + z1 is used)
  // light-curve front end (twk_magnify_lightcurve): when `t` is set, zeta = -(tau + i u0) e^{i alpha},
  // tau = (t - t0) / tE, is computed here from the epoch and the model's trajectory parameters; `zeta` is unused
  const double* t;           // [n_sources] epochs, or null
  const double* t0;          // [n_models]
  const double* u0;          // [n_models]
  const double* tE;          // [n_models]
  const double* alpha;       // [n_models]
  // lens orbital motion to first order (twk_magnify_lightcurve_orbital): s(t) = s + ds_dt (t - t0),
  // alpha(t) = alpha + dalpha_dt (t - t0); null = static lens
  const double* ds_dt;       // [n_models] or null
  const double* dalpha_dt;   // [n_models] or null
};

struct SourceParams {
  Lens L;
  cd zc;
  double rho;
  uint32_t status;   // TWK_ST_DOMAIN preset when outside P:374's range
  bool valid;
};

__device__ __forceinline__ SourceParams load_source(const Batch& b, long long src) {
  SourceParams P;
  const long long m_in = b.model_id ? (long long)b.model_id[src] : (b.n_models == 1 ? 0 : src);
  const long long m = (m_in >= 0 && m_in < b.n_models) ? m_in : 0;   // never read outside the model arrays
  double s = b.s[m];
  const double q = b.q[m], rho = b.rho[m];
  if (b.t) {
    const double dt = b.t[src] - b.t0[m];
    const double tau = dt / b.tE[m], u0 = b.u0[m];
    double alpha = b.alpha[m];
    if (b.ds_dt) {   // the lens of THIS epoch (what contour integration is preferred for)
      s = fma(b.ds_dt[m], dt, s);
      alpha = fma(b.dalpha_dt[m], dt, alpha);
    }
    double sa, ca;
    sincos(alpha, &sa, &ca);
    P.zc = mk(-(tau * ca - u0 * sa), -(tau * sa + u0 * ca));
  } else {
    P.zc = mk(b.zeta[2 * src], b.zeta[2 * src + 1]);
  }
  P.rho = rho;
  // finite, positive, and of a magnitude whose fourth powers stay finite (the coefficients are quartic in zeta and s)
  constexpr double kHuge = 1e50;
  P.valid = (s > 0.0) && (q > 0.0) && (rho > 0.0) && (s < kHuge) && (q < kHuge) && (rho < kHuge) && (fabs(P.zc.x) < kHuge) &&
            (fabs(P.zc.y) < kHuge) && (s > 1.0 / kHuge) && (q > 1.0 / kHuge) && m_in >= 0 && m_in < b.n_models;
  P.status = (P.valid && s >= 0.1 && s <= 10.0 && q >= 1e-9) ? 0u : 8u;
  P.L = make_lens(P.valid ? s : 1.0, P.valid ? q : 1.0);
  if (b.frame == 1) P.zc.x += P.L.z2 - P.L.s;   // z1 = -q s / (1 + q) = z2 - s  (reading F-1)
  return P;
}

// block-wide sum of two doubles over kWarps warps -- result valid in every thread
template <int kWarps = 2>
__device__ __forceinline__ void block_sum2(double& a, double& b, double* scratch /* >= 2 kWarps doubles */) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
  }
  const int warp = threadIdx.x >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) {
    scratch[2 * warp] = a;
    scratch[2 * warp + 1] = b;
  }
  __syncthreads();
  a = scratch[0];
  b = scratch[1];
#pragma unroll
  for (int w = 1; w < kWarps; ++w) {
    a += scratch[2 * w];
    b += scratch[2 * w + 1];
  }
}

// ------------------------------------------------------------------------------------------------------------
// Fixed-sampling mode.  TILE threads; records of one tile of samples in shared memory ([26][TILE]); the interval
// (j-1 -> j) is evaluated by the thread of sample j, with the previous tile's last record carried over.
// ------------------------------------------------------------------------------------------------------------
// SEEDED: every sample is solved as the adaptive kernels solve it -- centre_seeds() once per source, then the seeded
// Newton solve with Vieta recovery and the cold solver as fallback (twk_images_fixed_seeded; diag counts the events).
template <int TILE, bool SEEDED>
__global__ void __launch_bounds__(TILE) fixed_kernel(Batch b, int N, double* __restrict__ out_z, int8_t* __restrict__ out_kind,
                                                     int8_t* __restrict__ out_count, double* __restrict__ out_mu,
                                                     double* __restrict__ out_err, unsigned* __restrict__ diag) {
  extern __shared__ double sm[];
  double* rec = sm;                          // [26][TILE]
  double* carry = rec + kRecDoubles * TILE;  // [26] last record of the previous tile
  double* first = carry + kRecDoubles;       // [26] record of sample 0
  double* red = first + kRecDoubles;         // [2 * TILE/32]
  double* seeds = red + 2 * (TILE / 32);     // [31] seed block of the source (SEEDED)
  const int t = threadIdx.x;
  for (long long src = blockIdx.x; src < b.n_sources; src += gridDim.x) {
    const SourceParams S = load_source(b, src);
    if (!S.valid) {
      if (t == 0) {
        if (out_mu) out_mu[src] = nan("");
        if (out_err) out_err[src] = nan("");
      }
      continue;
    }
    double accA = 0.0, accE = 0.0;
    const double dth = kTwoPi / double(N);
    if (SEEDED) {
      if (t == 0) centre_seeds(S.L, S.zc, S.rho, seeds, 1);
      __syncthreads();
    }
    for (int base = 0; base < N; base += TILE) {
      const int j = base + t;
      const RecRef mine{rec + t, TILE};
      int flags = 0;
      if (j < N) {
        const size_t o = (size_t)src * N + j;
        double sn, cs;
        sincos(kTwoPi * double(j) / double(N), &sn, &cs);
        flags = point_solve_cs<true>(S.L, S.zc, S.rho, cs, sn, SEEDED ? seeds : nullptr, 1, mine, out_z ? out_z + o * 10 : nullptr,
                                     out_kind ? out_kind + o * 5 : nullptr, out_count ? out_count + o : nullptr, mine);
      }
      if (SEEDED && diag) {
        const unsigned act = __ballot_sync(0xffffffffu, j < N), rcv = __ballot_sync(0xffffffffu, flags & kPointRecovered),
                       cold = __ballot_sync(0xffffffffu, flags & kPointCold), grd = __ballot_sync(0xffffffffu, flags & kPointGuard);
        if ((t & 31) == 0) {
          if (act) atomicAdd(diag + 0, (unsigned)__popc(act));
          if (rcv) atomicAdd(diag + 1, (unsigned)__popc(rcv));
          if (cold) atomicAdd(diag + 2, (unsigned)__popc(cold));
          if (grd) atomicAdd(diag + 3, (unsigned)__popc(grd));
        }
      }
      __syncthreads();
      if (j < N && j >= 1) {
        const RecRef prev = (t > 0) ? RecRef{rec + t - 1, TILE} : RecRef{carry, 1};
        const Piece P = eval_interval(prev, mine, dth, 0.0, 0.5);   // slope detector off in fixed mode
        accA += P.dA;
        accE += P.err;
      }
      __syncthreads();
      if (j < N && (t == TILE - 1 || j == N - 1))
        for (int e = 0; e < kRecDoubles; ++e) carry[e] = mine.at(e);
      if (j == 0)
        for (int e = 0; e < kRecDoubles; ++e) first[e] = mine.at(e);
    }
    __syncthreads();
    if (t == 0) {   // closing interval (N-1 -> 0)
      const Piece P = eval_interval(RecRef{carry, 1}, RecRef{first, 1}, dth, 0.0, 0.5);
      accA += P.dA;
      accE += P.err;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      accA += __shfl_xor_sync(0xffffffffu, accA, o);
      accE += __shfl_xor_sync(0xffffffffu, accE, o);
    }
    if ((t & 31) == 0) {
      red[2 * (t >> 5)] = accA;
      red[2 * (t >> 5) + 1] = accE;
    }
    __syncthreads();
    if (t == 0) {
      double A = 0.0, E = 0.0;
      for (int w = 0; w < TILE / 32; ++w) {
        A += red[2 * w];
        E += red[2 * w + 1];
      }
      if (out_mu) out_mu[src] = A / (kPi * S.rho * S.rho);
      if (out_err) out_err[src] = E / fabs(A);
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------------------
// Parity harness: the Eq.(6) coefficients of the point source at zeta (twk_coeffs_eq6), one thread per source.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) coeffs_kernel(Batch b, double* __restrict__ out_c) {
  for (long long src = (long long)blockIdx.x * 128 + threadIdx.x; src < b.n_sources; src += (long long)gridDim.x * 128) {
    const SourceParams S = load_source(b, src);
    if (!S.valid) continue;
    cd c[6];
    coeffs_eq6(mk(S.zc.x - S.L.z2, S.zc.y), S.L.s, S.L.m2, c);
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      out_c[src * 12 + 2 * i] = c[i].x;
      out_c[src * 12 + 2 * i + 1] = c[i].y;
    }
  }
}

// ------------------------------------------------------------------------------------------------------------
// FP64 FMA throughput probe: 8 independent DFMA chains per thread.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dfma_probe_kernel(int iters, double* __restrict__ out) {
  double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 1e-3, a2 = a0 + 2e-3, a3 = a0 + 3e-3, a4 = a0 + 4e-3, a5 = a0 + 5e-3,
         a6 = a0 + 6e-3, a7 = a0 + 7e-3;
  const double m = 0.999999, c = 1e-7;
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  const double sum = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (sum == 123.456) out[0] = sum;   // never true; keeps the chains alive
}

}  // namespace twk
