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
  double slope_gate2;    // square of the slope detector's proximity gate (twk_options.slope_gate)
  double slope_cos2;     // square of the largest |cos| still counted as perpendicular (twk_options.slope_cos)
  int ps_test;           // N1: point-source adequacy tests in front of the contour path (twk_options.point_source_test)
  int group;             // sources per group, 1..64 (smaller for small batches: more CTAs get work)
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
constexpr int kS1Group = 64;      // sources per team and group (one centre solve per thread)

// Q teams of 64 threads per CTA.  A CTA takes a super-group of Q x 64 consecutive sources; team q owns sources
// q*64 .. q*64+63 of it and keeps its own shared-memory state; only the barriers are CTA-wide, which keeps the teams
// in step so that the warps of an SM run through the same ~35 KB of hot code together instead of streaming it at
// a dozen different places (instruction fetch was the top stall of the one-team kernel).
template <int Q>
__host__ __device__ constexpr size_t stage1_smem_bytes() {
  return (size_t)(Q * (kRecDoubles * kThreads + kSeedDoubles * kS1Group + kS1ParamRows * kS1Group + 2 * kS1Group) +
                  2 * Q * 4) * 8 +
         (size_t)(Q * 2 * kS1Group + 2 * Q * 2 + 2 * Q + 4) * 4 + Q * kS1Group;
}

template <int Q, int kMinBlocks>
__global__ void __launch_bounds__(Q * kThreads, kMinBlocks) stage1_kernel(Stage1Args p) {
  extern __shared__ double sm[];
  const int tid = threadIdx.x;
  const int q = tid >> 6, t = tid & (kThreads - 1), warp = (tid >> 5) & 1;
  double* recs_all = sm;                                                  // [Q][26][64]
  double* seeds_all = recs_all + Q * kRecDoubles * kThreads;              // [Q][30][64] seed blocks; column = source
  double* prm_all = seeds_all + Q * kSeedDoubles * kS1Group;              // [Q][8][64]
  double* res_mu_all = prm_all + Q * kS1ParamRows * kS1Group;             // [Q][64]
  double* res_err_all = res_mu_all + Q * kS1Group;                        // [Q][64]
  double* scratch = res_err_all + Q * kS1Group;                           // [2 (round parity)][Q][2 warps][2]
  int* res_ns_all = reinterpret_cast<int*>(scratch + 2 * Q * 4);          // [Q][64]
  int* res_st_all = res_ns_all + Q * kS1Group;                            // [Q][64]
  int* fscr = res_st_all + Q * kS1Group;                                  // [2][Q][2] flags of each warp
  int* slots = fscr + 2 * Q * 2;                                          // [2][Q] hand-over slot of each team's source
  int* iscr = slots + 2 * Q;                                              // [4]
  uint8_t* res_pend_all = reinterpret_cast<uint8_t*>(iscr + 4);           // [Q][64]
  double* recs = recs_all + q * kRecDoubles * kThreads;
  double* seeds = seeds_all + q * kSeedDoubles * kS1Group;
  double* prm = prm_all + q * kS1ParamRows * kS1Group;
  double* res_mu = res_mu_all + q * kS1Group;
  double* res_err = res_err_all + q * kS1Group;
  int* res_ns = res_ns_all + q * kS1Group;
  int* res_st = res_st_all + q * kS1Group;
  uint8_t* res_pend = res_pend_all + q * kS1Group;
  double cs, sn;
  sincospi(double(t) / 32.0, &sn, &cs);   // theta_t = 2 pi t / 64 (reading A-3)
  const RecRef mine{recs + t, kThreads};
  const RecRef next{recs + ((t + 1) & (kThreads - 1)), kThreads};
  const long long n = p.b.n_sources;
  const int G = p.group;
  const long long n_groups = (n + Q * G - 1) / (Q * G);   // super-groups
  int parity = 0;

  for (;;) {
    __syncthreads();
    if (tid == 0) iscr[0] = atomicAdd(p.cursor, 1);
    __syncthreads();
    const long long g = iscr[0];
    if (g >= n_groups) break;
    const long long base = (g * Q + q) * G;   // first source of this team
    // ---- phase 1: parameters and centre roots of source base + t --------------------------------------------------
    {
      const long long src = base + t;
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
          centre_seeds(S.L, S.zc, S.rho, seeds + t, kS1Group);
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
        }
        prm[7 * kS1Group + t] = code_as_double(code);
      }
    }
    __syncthreads();
    // ---- phase 2: one source per team at a time, one thread per boundary sample ---------------------------------------
    const int cnt = (int)((n - base < G) ? (n > base ? n - base : 0) : G);   // of this team
    for (int i = 0; i < G; ++i) {
      if (g * Q * G + i >= n) break;              // CTA-uniform: no team has a source i
      const int code = (i < cnt) ? code_of(prm[7 * kS1Group + i]) : 0;
      const bool active = (code & 256) != 0;            // team-uniform
      if (Q == 1 && !active) {                          // nothing to do for this source (CTA-uniform with one team)
        if (t == 0 && i < cnt && !(code & 512)) {       // invalid parameters: NaN out, status 8
          res_mu[i] = nan("");
          res_err[i] = nan("");
          res_ns[i] = 0;
          res_st[i] = 8;
          res_pend[i] = 0;
        }
        continue;
      }
      double rho = 1.0;
      int flags = 0;
      if (active) {
        Lens L;
        L.s = prm[0 * kS1Group + i];
        L.m1 = prm[1 * kS1Group + i];
        L.m2 = prm[2 * kS1Group + i];
        L.z2 = prm[3 * kS1Group + i];
        const cd zc = mk(prm[4 * kS1Group + i], prm[5 * kS1Group + i]);
        rho = prm[6 * kS1Group + i];
        flags = point_solve_cs(L, zc, rho, cs, sn, seeds + i, kS1Group, mine, nullptr, nullptr, nullptr);
      }
      __syncthreads();                                   // records of every team complete
      Piece P;
      double A, E;
      double* sc;
      int* fs;
      constexpr int kSlopeVote = 1 << 8;
      for (;;) {
        P.dA = 0.0;
        P.err = 0.0;
        P.crossing = 0;
        P.slope = 0;
        if (active) P = eval_interval(mine, next, kTwoPi / double(kThreads), p.slope_gate2, p.slope_cos2);
        // team sums: warp shuffle, then the two warps of the team through (double-buffered) shared memory
        A = P.dA;
        E = P.err;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
          A += __shfl_xor_sync(0xffffffffu, A, o);
          E += __shfl_xor_sync(0xffffffffu, E, o);
        }
        const int vote = (int)__reduce_or_sync(0xffffffffu, (unsigned)(flags | (P.slope ? kSlopeVote : 0)));
        sc = scratch + parity * (Q * 4);
        fs = fscr + parity * (Q * 2);
        if ((tid & 31) == 0) {
          sc[q * 4 + warp * 2] = A;
          sc[q * 4 + warp * 2 + 1] = E;
          fs[q * 2 + warp] = vote;
        }
        __syncthreads();
        int any = 0;
#pragma unroll
        for (int j = 0; j < 2 * Q; ++j) any |= fs[j];
        if (!(any & kSlopeVote)) break;                  // the common case: no extra barrier
        // a5, slope detector: re-judge the flagged real pairs as ghosts and evaluate the contour again.
        // A record is changed by one thread per phase: the interval on its left (creation into it) first, then the
        // interval on its right (annihilation out of it) if it still has five images.
        parity ^= 1;
        if (P.slope && P.crossing > 0) {
          demote_pair(next, P.slope & 15, (P.slope >> 4) & 15);
          flags |= kPointSlope;                          // reaches the team's flags through the next vote
        }
        __syncthreads();
        if (P.slope && P.crossing < 0 && mine.nreal() == 5) {
          demote_pair(mine, P.slope & 15, (P.slope >> 4) & 15);
          flags |= kPointSlope;
        }
        __syncthreads();
      }
      // every thread sees every team's sums: the decisions are CTA-uniform
      bool any_pend = false, pend = false, finite = true;
#pragma unroll
      for (int qq = 0; qq < Q; ++qq) {
        const double Aq = sc[qq * 4] + sc[qq * 4 + 2], Eq = sc[qq * 4 + 1] + sc[qq * 4 + 3];
        const bool act = ((g * Q + qq) * G + i < n) && (code_of(prm_all[(qq * kS1ParamRows + 7) * kS1Group + i]) & 256);
        const bool fin = isfinite(Aq) && isfinite(Eq);
        const bool pd = act && fin && !(Eq <= p.tol * fabs(Aq)) && !p.final_stage;   // stop rule P:272
        any_pend = any_pend || pd;
        if (qq == q) {
          A = Aq;
          E = Eq;
          pend = pd;
          finite = fin;
        }
      }
      flags = (fs[q * 2] | fs[q * 2 + 1]) & (kSlopeVote - 1);
      if (any_pend) {
        // a9: append to the refinement worklist; hand the first-iteration state over when a slot is free
        int* sl = slots + parity * Q;
        if (t == 0 && pend) {
          const int slot = atomicAdd(p.list_count, 1);
          p.list[slot] = (int32_t)(base + i);
          sl[q] = slot;
        }
        __syncthreads();
        if (pend) {
          const long long slot = sl[q];
          if (slot < p.handoff_slots) {
            double* h = p.handoff + (size_t)slot * kHandDoubles;
#pragma unroll
            for (int e = 0; e < kRecDoubles; ++e) h[e * kThreads + t] = mine.at(e);
            h[kRecDoubles * kThreads + t] = P.dA;
            h[(kRecDoubles + 1) * kThreads + t] = P.err;
            if (t < kSeedDoubles) h[(kRecDoubles + 2) * kThreads + t] = seeds[t * kS1Group + i];
          }
        }
      }
      if (t == 0 && i < cnt) {
        if (!active) {   // invalid parameters: NaN out, status 8 (done by the point-source tests: nothing to write)
          if (code & 512) {
          } else {
          res_mu[i] = nan("");
          res_err[i] = nan("");
          res_ns[i] = 0;
          res_st[i] = 8;
          res_pend[i] = 0;
          }
        } else {
          uint32_t status = (uint32_t)(code & 255);
          if (!finite) status |= 16u;
          else if (E <= p.tol * fabs(A)) status |= 1u;               // stop rule P:272
          else if (p.final_stage) status |= 2u;                       // cap P:326
          if (flags & kPointRepaired) status |= 4u;
          if (flags & kPointNonFinite) status |= 16u;
          if (flags & kPointSlope) status |= 32u;
          res_mu[i] = A * rcp(kPi * rho * rho);
          res_err[i] = E * rcp(fabs(A));
          res_ns[i] = kThreads;
          res_st[i] = (int)status;
          res_pend[i] = pend ? 1 : 0;
        }
      }
      parity ^= 1;
    }
    __syncthreads();
    // ---- phase 3: coalesced results -----------------------------------------------------------------------------------
    {
      const long long src = base + t;
      if (t < G && src < n && !res_pend[t]) {
        p.out_mu[src] = res_mu[t];
        if (p.out_err) p.out_err[src] = res_err[t];
        if (p.out_nsamples) p.out_nsamples[src] = res_ns[t];
        if (p.out_status) p.out_status[src] = (uint32_t)res_st[t];
      }
    }
  }
}

}  // namespace twk
