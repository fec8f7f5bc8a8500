// twk_stage1.cuh -- stage 1 of twk_magnify: the first iteration (64 uniform boundary samples) of EVERY source.
//
// One 64-thread CTA takes a group of 64 consecutive sources from an atomic cursor:
//   phase 1  thread i cold-solves the point source at the CENTRE of source i (Laguerre + deflation): its five
//            planet-frame roots and their first-order response to a source displacement are the seeds of that
//            source's boundary samples (centre_seeds(), twk_contour.cuh);
//   phase 2  for each source of the group: thread t solves boundary sample t by seeded Newton on the undeflated
//            quintic (verified; cold fallback), writes its record to shared memory, evaluates interval (t, t+1),
//            block-reduces area and error and applies the stop rule.  An unfinished source is appended to
//            the refinement worklist (a9) and its whole first-iteration state -- 64 records, 64 interval
//            pieces, seeds -- is handed to stage 2 through the hand-over arena (coalesced 512 B rows);
//   phase 3  coalesced write of the group's results.
// Per-source state of a finished source never leaves the SM: records [26][64], seeds [30][64], parameters [8][64].
#pragma once

#include "twk_kernels.cuh"

namespace twk {

struct Stage1Args {
  Batch b;
  double tol;
  int final_stage;       // 1: there is no refinement stage (max_samples < 128): cap status instead of pending
  int* cursor;           // group fetch counter (zeroed before launch)
  int32_t* list;         // [n_sources] a9: worklist of unfinished sources, appended in completion order
  int* list_count;       // entries of `list` (zeroed before launch)
  double* handoff;       // [handoff_slots][kHandDoubles] first-iteration state of worklist entries < handoff_slots
  long long handoff_slots;
  double* out_mu;
  double* out_err;       // may be null
  int32_t* out_nsamples; // may be null
  uint32_t* out_status;  // may be null
};

constexpr int kS1ParamRows = 8;   // s, m1, m2, z2, Re zc, Im zc, rho, status|valid
__host__ __device__ inline size_t stage1_smem_bytes() {
  return (size_t)(kRecDoubles * kThreads + kSeedDoubles * kThreads + kS1ParamRows * kThreads + 2 * kThreads + 8) * 8 +
         (size_t)(2 * kThreads + 4) * 4 + kThreads;
}

// block-wide sum of two doubles and OR of an int over 64 threads (2 warps); result valid in every thread
__device__ __forceinline__ void block_sum2_or(double& a, double& b, int& f, double* scratch /* >= 4 doubles */,
                                              int* iscratch /* >= 2 ints */) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
  }
  f = __reduce_or_sync(0xffffffffu, (unsigned)f);
  const int warp = threadIdx.x >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) {
    scratch[2 * warp] = a;
    scratch[2 * warp + 1] = b;
    iscratch[warp] = f;
  }
  __syncthreads();
  a = scratch[0] + scratch[2];
  b = scratch[1] + scratch[3];
  f = iscratch[0] | iscratch[1];
}

__global__ void __launch_bounds__(kThreads, 6) stage1_kernel(Stage1Args p) {
  extern __shared__ double sm[];
  double* recs = sm;                                   // [26][64]
  double* seeds = recs + kRecDoubles * kThreads;       // [30][64]: seed block (twk_contour.cuh); column = source
  double* prm = seeds + kSeedDoubles * kThreads;       // [8][64]
  double* res_mu = prm + kS1ParamRows * kThreads;      // [64]
  double* res_err = res_mu + kThreads;                 // [64]
  double* scratch = res_err + kThreads;                // [8]
  int* res_ns = reinterpret_cast<int*>(scratch + 8);   // [64]
  int* res_st = res_ns + kThreads;                     // [64]
  int* iscr = res_st + kThreads;                       // [4]
  uint8_t* res_pend = reinterpret_cast<uint8_t*>(iscr + 4);   // [64]

  const int t = threadIdx.x;
  double cs, sn;
  sincospi(double(t) / 32.0, &sn, &cs);   // theta_t = 2 pi t / 64 (reading A-3)
  const RecRef mine{recs + t, kThreads};
  const RecRef next{recs + ((t + 1) & (kThreads - 1)), kThreads};
  const long long n = p.b.n_sources;
  const long long n_groups = (n + kThreads - 1) / kThreads;

  for (;;) {
    __syncthreads();
    if (t == 0) iscr[0] = atomicAdd(p.cursor, 1);
    __syncthreads();
    const long long g = iscr[0];
    if (g >= n_groups) break;
    const long long base = g * kThreads;
    // ---- phase 1: parameters and centre roots of source base + t --------------------------------------------------
    {
      const long long src = base + t;
      if (src < n) {
        const SourceParams S = load_source(p.b, src);
        prm[0 * kThreads + t] = S.L.s;
        prm[1 * kThreads + t] = S.L.m1;
        prm[2 * kThreads + t] = S.L.m2;
        prm[3 * kThreads + t] = S.L.z2;
        prm[4 * kThreads + t] = S.zc.x;
        prm[5 * kThreads + t] = S.zc.y;
        prm[6 * kThreads + t] = S.rho;
        prm[7 * kThreads + t] = double((int)S.status | (S.valid ? 256 : 0));
        if (S.valid) centre_seeds(S.L, S.zc, S.rho, seeds + t, kThreads);
      }
    }
    __syncthreads();
    // ---- phase 2: one source at a time, one thread per boundary sample ------------------------------------------------
    const int cnt = (int)((n - base < kThreads) ? (n - base) : kThreads);
    for (int i = 0; i < cnt; ++i) {
      const int code = (int)prm[7 * kThreads + i];
      if (!(code & 256)) {   // invalid parameters: NaN out, status 8 (uniform branch)
        if (t == 0) {
          res_mu[i] = nan("");
          res_err[i] = nan("");
          res_ns[i] = 0;
          res_st[i] = 8;
          res_pend[i] = 0;
        }
        continue;
      }
      Lens L;
      L.s = prm[0 * kThreads + i];
      L.m1 = prm[1 * kThreads + i];
      L.m2 = prm[2 * kThreads + i];
      L.z2 = prm[3 * kThreads + i];
      const cd zc = mk(prm[4 * kThreads + i], prm[5 * kThreads + i]);
      const double rho = prm[6 * kThreads + i];
      int flags = point_solve_cs(L, zc, rho, cs, sn, seeds + i, kThreads, mine, nullptr, nullptr, nullptr);
      __syncthreads();
      const Piece P = eval_interval(mine, next, kTwoPi / double(kThreads));
      double A = P.dA, E = P.err;
      block_sum2_or(A, E, flags, scratch, iscr + 1);
      // every thread holds A, E: the decision is uniform
      const bool finite = isfinite(A) && isfinite(E);
      const bool pend = finite && !(E <= p.tol * fabs(A)) && !p.final_stage;   // stop rule P:272
      if (pend) {
        // a9: append to the refinement worklist; hand the first-iteration state over when a slot is free
        if (t == 0) {
          const int slot = atomicAdd(p.list_count, 1);
          p.list[slot] = (int32_t)(base + i);
          iscr[3] = slot;
        }
        __syncthreads();
        const long long slot = iscr[3];
        if (slot < p.handoff_slots) {
          double* h = p.handoff + (size_t)slot * kHandDoubles;
#pragma unroll
          for (int e = 0; e < kRecDoubles; ++e) h[e * kThreads + t] = mine.at(e);
          h[kRecDoubles * kThreads + t] = P.dA;
          h[(kRecDoubles + 1) * kThreads + t] = P.err;
          if (t < kSeedDoubles) h[(kRecDoubles + 2) * kThreads + t] = seeds[t * kThreads + i];
        }
      }
      if (t == 0) {
        uint32_t status = (uint32_t)(code & 255);
        if (!finite) status |= 16u;
        else if (E <= p.tol * fabs(A)) status |= 1u;               // stop rule P:272
        else if (p.final_stage) status |= 2u;                       // cap P:326
        if (flags & kPointRepaired) status |= 4u;
        if (flags & kPointNonFinite) status |= 16u;
        res_mu[i] = A / (kPi * rho * rho);
        res_err[i] = E / fabs(A);
        res_ns[i] = kThreads;
        res_st[i] = (int)status;
        res_pend[i] = pend ? 1 : 0;
      }
    }
    __syncthreads();
    // ---- phase 3: coalesced results -----------------------------------------------------------------------------------
    {
      const long long src = base + t;
      if (src < n) {
        if (!res_pend[t]) {
          p.out_mu[src] = res_mu[t];
          if (p.out_err) p.out_err[src] = res_err[t];
          if (p.out_nsamples) p.out_nsamples[src] = res_ns[t];
          if (p.out_status) p.out_status[src] = (uint32_t)res_st[t];
        }
      }
    }
  }
}

}  // namespace twk
