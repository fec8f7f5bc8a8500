// twk_stage1.cuh -- stage 1 of twk_magnify: the first iteration (64 uniform boundary samples) of EVERY source.
//
// One 64-thread CTA takes a group of up to 64 sources from an atomic cursor (consecutive sources in a batch of many waves; in
// a smaller batch blocks of 4 consecutive sources spread evenly over the batch -- the kSpread instance, see Stage1Args):
//   phase 1  thread i loads the parameters and the seed block of source i (stage 0: the five planet-frame roots of the
//            point source at the source's CENTRE and their first-order response to a source displacement);
//   phase 2  for each source of the group: thread t solves boundary sample t by seeded Newton on the undeflated
//            quintic (verified; cold fallback), writes its record to shared memory, evaluates interval (t, t+1),
//            block-reduces area and error and applies the stop rule.  An unfinished source is appended to
//            the refinement worklist (a9) and its whole first-iteration state -- 64 records, 64 interval
//            pieces, seeds -- is handed to stage 2 through the hand-over arena (coalesced 512 B rows);
//   phase 3  coalesced write of the group's results.
// With the point-source option (N1) phase 1 also runs the quadrupole and ghost-image tests; sources that pass
// are finished there.  Per-source state of a finished source never leaves the SM: records [26][64], seeds [31][64],
// parameters [8][64].
#pragma once

#include "twk_kernels.cuh"

namespace twk {

// ------------------------------------------------------------------------------------------------------------
// Stage 0: the point source at the CENTRE of every source (one thread per source): cold solve (Laguerre + deflation)
// and the first-order response of the five roots to a source displacement = the seed block of that source's boundary
// samples (centre_seeds(), twk_contour.cuh), written to the workspace as [kSeedDoubles][n_sources] so that stage 1 reads
// it coalesced.  A kernel of its own: the ~6 k instructions of the cold solver stay out of the instruction stream of
// the stage-1 loop (which fills the 32 KB instruction cache by itself).
// ------------------------------------------------------------------------------------------------------------
constexpr int kS0Threads = 128;
// 6 blocks per SM at 80 registers (measured 2 / 3 / 4 / 5 / 6 / 8 blocks per SM at 195 / 168 / 128 / 96 / 80 / 64 registers:
// 1.36 / 1.26 / 1.22 / 1.23 / 1.17 / 1.19 ms on config 3: the cold solver is one long dependent chain and wants warps more
// than it minds a few spills)
__global__ void __launch_bounds__(kS0Threads, 6) seeds_kernel(Batch b, double* __restrict__ seeds) {
  const long long n = b.n_sources;
  for (long long src = (long long)blockIdx.x * kS0Threads + threadIdx.x; src < n; src += (long long)gridDim.x * kS0Threads) {
    const SourceParams S = load_source(b, src);
    if (S.valid) centre_seeds(S.L, S.zc, S.rho, seeds + src, (int)0, n);
  }
}

struct Stage1Args {
  Batch b;
  double tol;
  double slope_gate2;    // square of the slope detector's proximity gate (twk_options.slope_gate)
  double slope_cos2;     // square of the largest |cos| still counted as perpendicular (twk_options.slope_cos)
  LinkConst K1;          // powers of the first iteration's interval width 2 pi / 64 (kernel parameters are constant-bank
                         // operands: no instruction materialises them)
  int ps_test;           // N1: point-source adequacy tests in front of the contour path (twk_options.point_source_test)
  int guard;             // L-4 guard: hidden-crossing term in the interval estimates (twk_options.hidden_crossing_guard)
  int group;             // sources per group, 1..64 (smaller for small batches: more CTAs get work)
  long long n_big;       // the first n_big groups have `group` sources, the rest of the batch goes out in groups of
  int tail_group;        // `tail_group` sources: the last wave of a large batch ends together
  int interleave;        // 1 (batches of a few waves at most): a group is made of blocks of 2^il_shift consecutive sources,
  int il_shift;          // the blocks n_big (= the number of groups) apart, instead of `group` consecutive sources:
                         // neighbouring sources -- the epochs of a light curve around its peak, the pixels of a map along
                         // a caustic -- are equally expensive, and with one or two groups per CTA the slowest CTA is the
                         // launch
  int final_stage;       // 1: there is no refinement stage (max_samples < 128): cap status instead of pending
  const double* seeds;   // [kSeedDoubles][n_sources] seed blocks written by stage 0
  int* cursor;           // group fetch counter (zeroed before launch)
  int32_t* list;         // [n_sources] a9: worklist of unfinished sources, appended in completion order
  int* list_count;       // entries of `list` (zeroed before launch)
  double* handoff;       // [handoff_slots][kHandDoubles] first-iteration state of worklist entries < handoff_slots
  long long handoff_slots;
  double* out_mu;        // may be null (twk_stage1_records)
  double* out_err;       // may be null
  int32_t* out_nsamples; // may be null
  uint32_t* out_status;  // may be null
  // diagnostics (twk_stage1_records): the 64 records of every source as this kernel computed them, and event counts
  double* dump;          // [n_sources][26][64] or null
  unsigned* diag;        // [4]: point solves, Vieta recoveries, cold solves, lens-guard hits; or null
};

constexpr int kS1ParamRows = 8;   // s, m1, m2, z2, Re zc, Im zc, rho, status|valid
constexpr int kS1Group = 64;      // sources per group at most (one centre solve per thread)
constexpr int kS1CtasPerSM = 6;   // 12 warps per SM at <= 168 registers (measured 3 / 4 / 5 / 6 CTAs: 42.8 / 34.9 / 32.5 / 29.8 ms)   // 12 warps per SM at <= 168 registers

__host__ __device__ constexpr size_t stage1_smem_bytes() {
  return (size_t)(kRecDoubles * kThreads + kSeedDoubles * kS1Group + kS1ParamRows * kS1Group + 2 * kS1Group + 2 * 4) * 8 +
         (size_t)(3 * kS1Group + 2 * 2 + 4) * 4 + kS1Group;
}

// kGuard: the L-4 hidden-crossing term (twk_options.hidden_crossing_guard) is compiled into its own instance of the
// kernel: the default instance carries no trace of it (the loop is sensitive to every extra instruction)
// kSpread: the groups of a batch of a few waves (Stage1Args::interleave), likewise an instance of its own: the instance
// that takes the large batches is the contiguous-group kernel and nothing else
template <bool kGuard, bool kSpread>
__global__ void __launch_bounds__(kThreads, kS1CtasPerSM) stage1_kernel(Stage1Args p) {
  extern __shared__ double sm[];
  double* recs = sm;                                          // [26][64] records of the current source
  double* seeds = recs + kRecDoubles * kThreads;              // [31][64] seed blocks; column = source of the group
  double* prm = seeds + kSeedDoubles * kS1Group;              // [8][64]  parameters; column = source of the group
  double* res_mu = prm + kS1ParamRows * kS1Group;             // [64]
  double* res_err = res_mu + kS1Group;                        // [64]
  double* scratch = res_err + kS1Group;                       // [2 (round parity)][2 warps][2] partial sums
  int* res_ns = reinterpret_cast<int*>(scratch + 2 * 4);      // [64]
  int* res_st = res_ns + kS1Group;                            // [64]
  int* res_src = res_st + kS1Group;                           // [64] source index of every column
  int* fscr = res_src + kS1Group;                             // [2 (round parity)][2 warps] flags + slope vote
  int* iscr = fscr + 2 * 2;                                   // [4]: group, -, -, hand-over slot
  uint8_t* res_pend = reinterpret_cast<uint8_t*>(iscr + 4);   // [64]

  const int t = threadIdx.x, warp = t >> 5;
  double cs, sn;
  sincospi(double(t) / 32.0, &sn, &cs);   // theta_t = 2 pi t / 64 (reading A-3)
  const RecRef mine{recs + t, kThreads};
  const RecRef next{recs + ((t + 1) & (kThreads - 1)), kThreads};
  const long long n = p.b.n_sources;
  constexpr bool il = kSpread;
  const long long n_big = p.n_big, n_in_big = n_big * p.group;
  const long long n_groups = il ? n_big : n_big + (n - n_in_big + p.tail_group - 1) / p.tail_group;
  int parity = 0;

  for (;;) {
    __syncthreads();
    if (t == 0) iscr[0] = atomicAdd(p.cursor, 1);
    __syncthreads();
    const long long g = iscr[0];
    if (g >= n_groups) break;
    const int G = (il || g < n_big) ? p.group : p.tail_group;
    const long long base = (g < n_big) ? g * p.group : n_in_big + (g - n_big) * p.tail_group;   // first source of the group
    // source of column `col` of the group (phase 2 reads it from res_src)
    auto src_at = [&](int col) -> long long {
      return il ? ((g + (long long)(col >> p.il_shift) * n_groups) << p.il_shift) + (col & ((1 << p.il_shift) - 1)) : base + col;
    };
    // ---- phase 1: parameters and centre roots of source base + t --------------------------------------------------
    {
      const long long src = src_at(t);
      if (il && t < G) {
        res_src[t] = (int)src;
        if (src >= n) prm[7 * kS1Group + t] = code_as_double(0);   // no source in this column (phase 2 skips it)
      }
      if (t < G && src < n) {
        const SourceParams S = load_source(p.b, src);
        prm[0 * kS1Group + t] = S.L.s;
        prm[1 * kS1Group + t] = S.L.m1;
        prm[2 * kS1Group + t] = S.L.m2;
        prm[3 * kS1Group + t] = S.L.z2;
        prm[4 * kS1Group + t] = S.zc.x;
        prm[5 * kS1Group + t] = S.zc.y;
        prm[6 * kS1Group + t] = S.rho;
        int code = (int)S.status | (S.valid ? 256 : 0);
        if (S.valid) {
          {   // all 31 loads in flight at once (one DRAM latency per group, not 31)
            double sv[kSeedDoubles];
#pragma unroll
            for (int e = 0; e < kSeedDoubles; ++e) sv[e] = __ldg(p.seeds + (size_t)e * (size_t)n + (size_t)src);
#pragma unroll
            for (int e = 0; e < kSeedDoubles; ++e) seeds[e * kS1Group + t] = sv[e];
          }
          if (p.ps_test) {   // N1: quadrupole + ghost-image tests; adequate -> no contour for this source
            const PsResult r = point_source_adequate_cold(S.L, S.zc, S.rho, seeds + t, kS1Group, p.tol);
            if (r.ok) {
              res_mu[t] = r.mu;
              res_err[t] = r.qrel;
              res_ns[t] = 0;
              res_st[t] = (int)(S.status | 1u | 64u);
              res_pend[t] = 0;
              code = (code & ~256) | 512;   // done: phase 2 skips it
            }
          }
        } else {             // invalid parameters: NaN out, status 8
          res_mu[t] = nan("");
          res_err[t] = nan("");
          res_ns[t] = 0;
          res_st[t] = 8;
          res_pend[t] = 0;
        }
        prm[7 * kS1Group + t] = code_as_double(code);
      }
    }
    __syncthreads();
    // ---- phase 2: one source at a time, one thread per boundary sample ------------------------------------------------
    const int cnt = il ? G : (int)((n - base < G) ? (n - base) : G);
    for (int i = 0; i < cnt; ++i) {
      const int code = code_of(prm[7 * kS1Group + i]);
      if (!(code & 256)) continue;                       // invalid or already done (uniform)
      Lens L;
      L.s = prm[0 * kS1Group + i];
      L.m1 = prm[1 * kS1Group + i];
      L.m2 = prm[2 * kS1Group + i];
      L.z2 = prm[3 * kS1Group + i];
      const cd zc = mk(prm[4 * kS1Group + i], prm[5 * kS1Group + i]);
      const double rho = prm[6 * kS1Group + i];
      int flags = point_solve_cs<true>(L, zc, rho, cs, sn, seeds + i, kS1Group, mine, nullptr, nullptr, nullptr, mine);
      if (p.diag) {
        const unsigned rec = __ballot_sync(0xffffffffu, flags & kPointRecovered), cold = __ballot_sync(0xffffffffu, flags & kPointCold),
                       grd = __ballot_sync(0xffffffffu, flags & kPointGuard);
        if ((t & 31) == 0) {
          atomicAdd(p.diag + 0, 32u);
          if (rec) atomicAdd(p.diag + 1, (unsigned)__popc(rec));
          if (cold) atomicAdd(p.diag + 2, (unsigned)__popc(cold));
          if (grd) atomicAdd(p.diag + 3, (unsigned)__popc(grd));
        }
      }
      __syncthreads();                                   // the 64 records are complete
      Piece P;
      double A, E;
      constexpr int kSlopeVote = 1 << 8;
      for (;;) {
        P = eval_interval(mine, next, p.K1, p.slope_gate2, p.slope_cos2);
        if (kGuard && P.crossing == 0) {
          const double h = kTwoPi / double(kThreads);
          P.err += hidden_crossing_term(RecRef{recs + ((t + kThreads - 1) & (kThreads - 1)), kThreads}, mine, next,
                                        RecRef{recs + ((t + 2) & (kThreads - 1)), kThreads}, h, h, h);
        }
        // sums: warp shuffle, then the two warps through (double-buffered) shared memory
        A = P.dA;
        E = P.err;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          A += __shfl_xor_sync(0xffffffffu, A, o);
          E += __shfl_xor_sync(0xffffffffu, E, o);
        }
        const int vote = (int)__reduce_or_sync(0xffffffffu, (unsigned)(flags | (P.slope ? kSlopeVote : 0)));
        double* sc = scratch + parity * 4;
        int* fs = fscr + parity * 2;
        if ((t & 31) == 0) {
          sc[warp * 2] = A;
          sc[warp * 2 + 1] = E;
          fs[warp] = vote;
        }
        __syncthreads();
        A = sc[0] + sc[2];
        E = sc[1] + sc[3];
        flags = fs[0] | fs[1];
        parity ^= 1;
        if (!(flags & kSlopeVote)) break;                // the common case: no extra barrier
        // a5, slope detector: re-judge the flagged real pairs as ghosts and evaluate the contour again.
        // A record is changed by one thread per phase: the interval on its left (creation into it) first, then the
        // interval on its right (annihilation out of it) if it still has five images.
        flags &= kSlopeVote - 1;
        if (P.slope && P.crossing > 0) {
          demote_pair(next, P.slope & 15, (P.slope >> 4) & 15);
          flags |= kPointSlope;                          // reaches every thread through the next vote
        }
        __syncthreads();
        if (P.slope && P.crossing < 0 && mine.nreal() == 5) {
          demote_pair(mine, P.slope & 15, (P.slope >> 4) & 15);
          flags |= kPointSlope;
        }
        __syncthreads();
      }
      if (p.dump) {
        double* d = p.dump + (size_t)(il ? (long long)res_src[i] : base + i) * (kRecDoubles * kThreads);
#pragma unroll 1
        for (int e = 0; e < kRecDoubles; ++e) d[e * kThreads + t] = mine.at(e);
      }
      // every thread holds A, E and the flags: the decisions are uniform
      const bool finite = isfinite(A) && isfinite(E);
      const bool pend = finite && !(E <= p.tol * fabs(A)) && !p.final_stage;   // stop rule P:272
      if (pend) {
        // a9: append to the refinement worklist; hand the first-iteration state over when a slot is free
        // Is ONE more iteration (64 samples where the error is) likely to finish this source?  If the error sits in
        // N_eff = E^2 / sum e_i^2 intervals, each gets ~64 / N_eff new samples and its error falls by about the square of
        // that: predicted E / (1 + 64 sum e_i^2 / E^2)^2.  A source whose prediction is still above 1.5 tolerances (error
        // spread evenly at a tight tolerance) is marked (sign bit of its worklist entry): stage 1.5 leaves it to stage 2.
        double q2 = P.err * P.err;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) q2 += __shfl_xor_sync(0xffffffffu, q2, o);
        double* sq = scratch + parity * 4;   // (the half of the double buffer the NEXT reduction will use: free now)
        if ((t & 31) == 0) sq[warp] = q2;
        if (t == 0) {
          const int slot = atomicAdd(p.list_count, 1);
          TWK_CHECK(slot >= 0 && slot < n, 4);
          iscr[3] = slot;
        }
        __syncthreads();
        const long long slot = iscr[3];
        if (t == 0) {
          const double S2 = sq[0] + sq[1], E2 = E * E, den = E2 + 64.0 * S2;
          const bool spread = E * E2 * E2 > 1.5 * p.tol * fabs(A) * den * den;   // E / (1 + 64 S2 / E^2)^2 > 1.5 tol |A|
          p.list[slot] = (int32_t)(il ? (long long)res_src[i] : base + i) | (spread ? (int32_t)0x80000000 : 0);
        }
        if (slot < p.handoff_slots) {
          double* h = p.handoff + (size_t)slot * kHandDoubles;
#pragma unroll
          for (int e = 0; e < kRecDoubles; ++e) h[e * kThreads + t] = mine.at(e);
          h[kRecDoubles * kThreads + t] = P.dA;
          h[(kRecDoubles + 1) * kThreads + t] = P.err;
          if (t < kSeedDoubles) h[(kRecDoubles + 2) * kThreads + t] = seeds[t * kS1Group + i];
          if (t >= 32 && t < 32 + 9) {   // header: what stage 2 needs to start this source without looking anything up
            const int k = t - 32;
            h[kHandHeader + k] = (k == 0) ? __longlong_as_double(il ? (long long)res_src[i] : base + i)
                                          : (k == 8) ? code_as_double(code & 255) : prm[(k - 1) * kS1Group + i];
          }
        }
      }
      if (t == 0) {
        uint32_t status = (uint32_t)(code & 255);
        if (!finite) status |= 16u;
        else if (E <= p.tol * fabs(A)) status |= 1u;               // stop rule P:272
        else if (p.final_stage) status |= 2u;                       // cap P:326
        if (flags & kPointRepaired) status |= 4u;
        if (flags & (kPointNonFinite | kPointGuard)) status |= 16u;
        if (flags & kPointSlope) status |= 32u;
        res_mu[i] = A * rcp(kPi * rho * rho);
        res_err[i] = E * rcp(fabs(A));
        res_ns[i] = kThreads;
        res_st[i] = (int)status;
        res_pend[i] = pend ? 1 : 0;
      }
    }
    __syncthreads();
    // ---- phase 3: coalesced results -----------------------------------------------------------------------------------
    {
      const long long src = src_at(t);
      if (t < G && src < n && !res_pend[t] && p.out_mu) {
        p.out_mu[src] = res_mu[t];
        if (p.out_err) p.out_err[src] = res_err[t];
        if (p.out_nsamples) p.out_nsamples[src] = res_ns[t];
        if (p.out_status) p.out_status[src] = (uint32_t)res_st[t];
      }
    }
  }
}

}  // namespace twk
