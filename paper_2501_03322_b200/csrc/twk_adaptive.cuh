// twk_adaptive.cuh -- a8 + a9: the adaptive contour loop for one source per CTA (refinement stages 2 and 3; see
// twk_kernels.cuh).  Every iteration adds up to 64 new samples, one thread each; stage 2 runs 64-thread CTAs, stage 3
// 128-thread CTAs whose extra warps share the O(n) passes over the sorted state.  A stage-2 source normally arrives with
// its first iteration done: stage 1 handed over its 64 records, 64 interval pieces and seed block (hand-over arena),
// which are used in place; without a free hand-over slot the first iteration is recomputed here.  A source that fills
// stage 2's capacity takes its whole state along to stage 3 (carry-over arena) and continues there; without a free
// carry-over slot stage 3 recomputes it from its first sample.  New samples are solved by seeded Newton from the source
// centre's seed block, with the cold solver as verified fallback.
#pragma once

#include "twk_kernels.cuh"

namespace twk {

// eval_interval as an out-of-line call: used only by the slope detector's repair pass (rare), kept out of the hot
// instruction stream
TWK_NOINLINE Piece eval_interval_cold(RecRef A, RecRef B, double dth, double slope_gate2, double slope_cos2) {
  return eval_interval(A, B, dth, slope_gate2, slope_cos2);
}

// Stage 2 -> stage 3 carry-over of a source that filled stage 2's capacity (rare: out of line).  Slot layout: carry_doubles().
// Records of id < 64 of a handed-over source are still in its hand-over slot ([26][64]), the others in the CTA's arena.
TWK_NOINLINE void carry_out(double* cs, int C, int n, const double* theta, const double* dA, const double* er,
                            const uint16_t* ids, const double* arena, const double* hand, int status_bits) {
  const int t = threadIdx.x;
  for (int id = t; id < n; id += blockDim.x) {
    const RecRef r = (hand && id < 64) ? RecRef{const_cast<double*>(hand) + id, 64}
                                       : RecRef{const_cast<double*>(arena) + (size_t)id * kRecDoubles, 1};
    double* d = cs + (size_t)id * kRecDoubles;
#pragma unroll 2
    for (int e = 0; e < kRecDoubles; ++e) d[e] = r.at(e);
  }
  double* cth = cs + (size_t)C * kRecDoubles;
  uint16_t* cid = reinterpret_cast<uint16_t*>(cth + 3 * (size_t)C);
  for (int i = t; i < n; i += blockDim.x) {
    cth[i] = theta[i];
    cth[C + i] = dA[i];
    cth[2 * C + i] = er[i];
    cid[i] = ids[i];
  }
  if (t == 0) {
    double* hd = cs + (size_t)C * (kRecDoubles + 3) + C / 4;
    hd[0] = code_as_double(n);
    hd[1] = code_as_double(status_bits);
  }
}

struct AdaptArgs {
  Batch b;
  double tol;
  double slope_gate2;    // square of the slope detector's proximity gate (twk_options.slope_gate)
  double slope_cos2;     // square of the largest |cos| still counted as perpendicular (twk_options.slope_cos)
  int cap;               // sample capacity of this stage (<= 4096)
  int subtract_avg_tol;
  int guard;             // L-4 guard: hidden-crossing term in the interval estimates (twk_options.hidden_crossing_guard)
  int final_stage;       // 1: cap reached -> return value + estimate with TWK_ST_CAP; 0: hand to next stage
  const int32_t* remap;  // stage 2 behind stage 1.5: worklist of ENTRIES (indices into `list` and the hand-over arena) that are
                         // still to be refined; null: entries 0 .. count - 1 in order
  const int32_t* list;   // worklist of source ids (null: all sources 0..n_sources-1)
  const int* count;      // number of entries of `list` (device; null: n_sources)
  int* cursor;           // dynamic work fetch counter (device, zeroed before launch)
  int32_t* next_list;    // stage 2 only: sources that need stage 3 ...
  int* next_count;       // ... appended with atomicAdd
  double* arena;         // stages 2/3: gridDim.x * cap records of kRecDoubles doubles
  const double* seeds;   // [kSeedDoubles][n_sources] seed blocks written by stage 0
  const double* handoff; // stage 2: hand-over arena written by stage 1 (null: recompute the first iteration)
  long long handoff_slots;   // worklist entries < handoff_slots have a hand-over slot
  // carry-over arena between the refinement stages: a source that fills stage 2's capacity takes its whole state along
  // (records, sorted angles, interval pieces) instead of being recomputed from its first sample by stage 3
  double* carry;         // [carry_slots][carry_doubles(carry_cap)] or null
  long long carry_slots; // entries of the next stage's worklist < carry_slots have a slot
  int carry_cap;         // sample capacity of a slot (= stage 2's cap)
  int carry_role;        // 0 none, 1 this stage writes slots (stage 2), 2 this stage reads them (stage 3)
  double* out_mu;
  double* out_err;       // may be null
  int32_t* out_nsamples; // may be null
  uint32_t* out_status;  // may be null
};

// carry-over slot, in doubles: records [C][26] | theta [C] | dA [C] | err [C] | ids [C] u16 | header [8]: n, status bits
__host__ __device__ inline size_t carry_doubles(int C) { return (size_t)C * (kRecDoubles + 3) + (size_t)C / 4 + 8; }
constexpr int kScrDoubles = 20;   // per-thread scratch of point_solve_cs<true> (roots and residuals of the five roots)
__host__ __device__ inline size_t adaptive_smem_bytes(int cap, bool scr, bool tile, int threads = kThreads) {
  // (with a tile the scratch of the point solves is the tile column the record goes to)
  size_t doubles = 3 * (size_t)cap + 2 * kThreads + (threads > kThreads ? 16 : 8) + 32 + (scr && !tile ? kScrDoubles * kThreads : 0) + (tile ? kRecDoubles * kThreads : 0);
  size_t ints = 2 * kThreads + 8;
  return doubles * 8 + ints * 4 + (size_t)cap * 2;
}

// 6 CTAs per SM (168 registers): measured 4 / 5 / 6 / 8 CTAs per SM on configs 3 and 5: 9.4 / 9.3 / 8.6 / 8.8 ms and
// 7.6 / 7.4 / 6.7 / 7.0 ms -- the kernel is latency-bound and wants warps, but at 128 registers it spills
// kGuard: the L-4 hidden-crossing term lives in its own instance of the kernel (see stage1_kernel)
// kScr:   [20][64] doubles of shared-memory scratch for the residual detector (stage 2; at the 4096-sample capacity of
//         stage 3 the 10 KB would cost the second resident CTA, so that instance selects in registers)
// kTile:  the records of the iteration's NEW samples are written twice, to the arena (where later iterations find them) and
//         to a [26][64] shared-memory tile; the interval evaluations of the same iteration read every new record -- each
//         thread's own, above all -- from the tile instead of waiting for the arena
// TB:     threads per CTA.  64 = one thread per new sample (stage 2).  Stage 3 runs 128: the 64 new samples of an iteration
//         are solved and their intervals evaluated by the first two warps as before, but the O(n) passes over the sorted
//         state (sums, weight scan, shift) that dominate an iteration at thousands of samples are shared by four warps
//         -- its 106 KB of shared memory allow two CTAs per SM whatever their width
template <bool kGuard, bool kScr, bool kTile, int TB>
__global__ void __launch_bounds__(TB, TB == kThreads ? 6 : 2) adaptive_kernel(AdaptArgs p) {
  static_assert(TB % 32 == 0 && TB >= kThreads && TB <= 256, "TB");
  constexpr int kWarps = TB / 32;
  // "one of the 64 threads that own a new sample": always true at compile time when the CTA has no others
#define TWK_FIRST64(tt) (TB == kThreads || (tt) < kThreads)
  extern __shared__ double sm[];
  const int cap = p.cap;
  double* theta = sm;            // [cap] sorted sample angles
  double* dA = theta + cap;      // [cap] area piece of interval (i, i+1)
  double* er = dA + cap;         // [cap] error piece of interval (i, i+1)
  double* newth = er + cap;      // [64]  angle of quantile k
  double* cth = newth + kThreads;   // [64] compacted new angles
  constexpr int kScanAt = (kWarps == 2) ? 4 : 8;   // scratch: block sums [0 .. 2 kWarps), warp totals of the scan behind them
  double* scratch = cth + kThreads; // [8] (two warps) or [16]
  double* seeds = scratch + 2 * kScanAt;   // [30 (+2)] seed block of the source (twk_contour.cuh)
  double* scrbuf = seeds + 32;      // [20][64] (kScr) scratch of the point solves
  double* tile = scrbuf + (kScr && !kTile ? kScrDoubles * kThreads : 0);   // [26][64] (kTile) records of this iteration's new samples
  int* newint = reinterpret_cast<int*>(tile + (kTile ? kRecDoubles * kThreads : 0));   // [64] interval of quantile k
  int* cint = newint + kThreads;    // [64] compacted
  int* iscr = cint + kThreads;      // [8]: current entry, two warp counts, slope count, -, carry-over slot
  uint16_t* ids = reinterpret_cast<uint16_t*>(iscr + 8);   // [cap] arena id of the sample at each sorted position

  const int t = threadIdx.x;
  const int lane = t & 31, warp = t >> 5;
  double* arena = p.arena + (size_t)blockIdx.x * (size_t)cap * kRecDoubles;
  // record of sample id: ids 0..63 of a handed-over source live in its hand-over slot ([26][64]), the rest in the arena
  const double* hand = nullptr;
  const double* carried = nullptr;   // stage 3: records 0 .. n_carried - 1 of a carried-over source live in its slot
  int n_carried = 0;
  int tile_base = 1 << 30;   // ids >= tile_base are in the tile (the current iteration's new samples)
  auto recref = [&](int id) -> RecRef {
    TWK_CHECK(id >= 0 && id < cap, 0);
    if (kTile && id >= tile_base) return RecRef{tile + (id - tile_base), kThreads};
    if (hand && id < kThreads) return RecRef{const_cast<double*>(hand) + id, kThreads};
    if (id < n_carried) return RecRef{const_cast<double*>(carried) + (size_t)id * kRecDoubles, 1};
    return RecRef{arena + (size_t)id * kRecDoubles, 1};
  };
  // L-4 guard term of interval (i, i + 1) in a sorted list of nn samples (neighbours i - 1 and i + 2, cyclic)
  auto guard_term = [&](int i, int nn) -> double {
    const int im = (i > 0) ? i - 1 : nn - 1, ib = (i + 1 < nn) ? i + 1 : 0, ip = (ib + 1 < nn) ? ib + 1 : 0;
    const double dm = (i > 0) ? theta[i] - theta[im] : kTwoPi - theta[im] + theta[i];
    const double d = (i + 1 < nn) ? theta[ib] - theta[i] : kTwoPi - theta[i] + theta[ib];
    const double dp = (ib + 1 < nn) ? theta[ip] - theta[ib] : kTwoPi - theta[ib] + theta[ip];
    return hidden_crossing_term(recref(ids[im]), recref(ids[i]), recref(ids[ib]), recref(ids[ip]), dm, d, dp);
  };
  const long long total = p.count ? (long long)*p.count : p.b.n_sources;

  // work fetch one source ahead: thread 0 takes the NEXT entry of the cursor at the start of the current source and
  // publishes it at its end, so the atomic's round trip is never waited for
  if (t == 0) iscr[0] = atomicAdd(p.cursor, 1);
  for (;;) {
    __syncthreads();
    const long long cur = iscr[0];
    if (cur >= total) break;
    int next_cur = 0;
    if (t == 0) next_cur = atomicAdd(p.cursor, 1);
    // a handed-over source starts from its slot's header; otherwise worklist -> model -> parameters
    const long long ent = p.remap ? (long long)p.remap[cur] : cur;
    hand = (p.handoff && ent < p.handoff_slots) ? p.handoff + (size_t)ent * kHandDoubles : nullptr;
    long long src;
    SourceParams S;
    if (hand) {
      const double* hd = hand + kHandHeader;
      src = __double_as_longlong(hd[0]);
      S.L.s = hd[1];
      S.L.m1 = hd[2];
      S.L.m2 = hd[3];
      S.L.z2 = hd[4];
      S.zc = mk(hd[5], hd[6]);
      S.rho = hd[7];
      S.status = (uint32_t)code_of(hd[8]);
      S.valid = true;
    } else {
      src = p.list ? (long long)(p.list[ent] & 0x7fffffff) : ent;   // (the sign bit is stage 1's note for stage 1.5)
      S = load_source(p.b, src);
    }
    TWK_CHECK(src >= 0 && src < p.b.n_sources, 4);
    if (t == 0) TWK_DEBUG_COUNT(6);
    if (!S.valid) {
      if (t == 0) {
        p.out_mu[src] = nan("");
        if (p.out_err) p.out_err[src] = nan("");
        if (p.out_nsamples) p.out_nsamples[src] = 0;
        if (p.out_status) p.out_status[src] = 8u;
      }
      __syncthreads();
      if (t == 0) iscr[0] = next_cur;
      continue;
    }
    // ---- first iteration: 64 uniform samples theta_j = 2 pi j / 64 (reading A-3) ----------------------
    int flags = 0;
    int n = 0;
    if (hand) {   // done by stage 1: take its interval pieces and seed block, use its records in place
      // the slot was written long ago (4 GB of hand-over traffic per call has left the L2): pull its 14.7 KB back
      // into the L2 now, the first solve hides the DRAM latency of the records
      {
        const char* hb = reinterpret_cast<const char*>(hand);
        asm volatile("prefetch.global.L2 [%0];" ::"l"(hb + t * 128));
        if (TB == kThreads && (t + kThreads) * 128 < kHandDoubles * 8)
          asm volatile("prefetch.global.L2 [%0];" ::"l"(hb + (t + kThreads) * 128));
      }
      if (TWK_FIRST64(t)) {
        theta[t] = kTwoPi * double(t) / double(kThreads);
        ids[t] = (uint16_t)t;
        dA[t] = hand[kRecDoubles * kThreads + t];
        er[t] = hand[(kRecDoubles + 1) * kThreads + t];
        flags |= recref(t).point_flags();
      }
      if (t < kSeedDoubles) seeds[t] = hand[(kRecDoubles + 2) * kThreads + t];
      n = kThreads;
    } else {      // not handed over: the loop below starts by inserting the 64 uniform samples into the empty list
      if (t < kSeedDoubles) seeds[t] = p.seeds[(size_t)t * (size_t)p.b.n_sources + (size_t)src];
    }
    uint32_t status = S.status;
    carried = nullptr;
    n_carried = 0;
    // (compile-time roles: the stage-2 instance of the kernel is the one with the tile and only writes slots, the
    //  stage-3 instance only reads them; neither carries the other's code)
    if (!kTile && p.carry_role == 2 && cur < p.carry_slots) {   // carried over from stage 2: continue where it stopped
      const int C = p.carry_cap;
      const double* cs = p.carry + (size_t)cur * carry_doubles(C);
      const double* hd = cs + (size_t)C * (kRecDoubles + 3) + C / 4;
      n = code_of(hd[0]);
      status |= (uint32_t)code_of(hd[1]);
      carried = cs;
      n_carried = n;
      const double* cth_ = cs + (size_t)C * kRecDoubles;
      const uint16_t* cid = reinterpret_cast<const uint16_t*>(cth_ + 3 * (size_t)C);
      for (int i = t; i < n; i += TB) {
        theta[i] = cth_[i];
        dA[i] = cth_[C + i];
        er[i] = cth_[2 * C + i];
        ids[i] = cid[i];
      }
    }
    bool exhausted = false, slope_seen = false;
    double A = 0.0, E = 0.0;
    for (;;) {
      __syncthreads();
      int m = kThreads;
      if (n == 0) {
        if (TWK_FIRST64(t)) {
          cth[t] = kTwoPi * double(t) / double(kThreads);
          cint[t] = -1;
        }
        __syncthreads();
      } else {
        // ---- area and error sums over all intervals (a7 reduction) ----------------------------------------------
        double a = 0.0, e = 0.0;
        for (int i = t; i < n; i += TB) {
          a += dA[i];
          e += er[i];
        }
        block_sum2<kWarps>(a, e, scratch);
        A = a;
        E = e;
        const double tolA = p.tol * fabs(A);
        if (!(isfinite(A) && isfinite(E))) { status |= 16u; break; }
        if (E <= tolA) { status |= 1u; break; }                       // stop rule P:272, reading A-1
        if (n + kThreads > cap) { exhausted = true; break; }          // cap P:326, reading A-6
        // ---- a8: error-weighted inverse-transform sampling, 64 quantiles ---------------------------
        const double avg = p.subtract_avg_tol ? tolA / double(n) : 0.0;   // "average tolerance", reading A-5
        double W = 0.0, unused = 0.0;
        for (int i = t; i < n; i += TB) W += fmax(er[i] - avg, 0.0);
        block_sum2<kWarps>(W, unused, scratch);
        const bool raw = !(W > 0.0);
        if (raw) W = E;
        const double scale = double(kThreads) / W;
        // Each interval marks the first quantile it owns (cint: interval | one-past-last quantile << 16, cth: its
        // exclusive cumulative weight); afterwards every quantile finds its owner by a max-scan over the marks and
        // computes its own angle: 64 angles in parallel even when one interval owns them all.
        if (TWK_FIRST64(t)) cint[t] = -1;
        double carry = 0.0;
        __syncthreads();
        for (int base = 0; base < n; base += TB) {
          const int i = base + t;
          const double w = (i < n) ? (raw ? er[i] : fmax(er[i] - avg, 0.0)) : 0.0;
          double x = w;   // inclusive scan over the 64 threads
  #pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const double y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
          }
          __syncthreads();
          if (lane == 31) scratch[kScanAt + warp] = x;
          __syncthreads();
          // prefix of the warps before this one, accumulated left to right: P_0 = 0, P_w = P_{w-1} + total_{w-1}
          double before = 0.0, whole = 0.0;
          if (kWarps == 2) {
            const double w0 = scratch[kScanAt], w1 = scratch[kScanAt + 1];
            if (warp == 1) before = w0;
            whole = w0 + w1;
          } else {
#pragma unroll
            for (int w2 = 0; w2 < kWarps; ++w2) {
              if (w2 == warp) before = whole;
              whole += scratch[kScanAt + w2];
            }
          }
          const double cum_incl = carry + (x + before);
          double cum_excl = __shfl_up_sync(0xffffffffu, cum_incl, 1);
          // bitwise the left neighbour's cum_incl: the last lane of the warp before holds x = total_{w-1}, and
          // total_{w-1} + P_{w-1} = P_w by construction (addition commutes exactly)
          if (lane == 0) cum_excl = carry + before;
          if (w > 0.0) {
            // quantile k has target (k + 1/2)/64 * W (reading A-4); this interval owns those in [cum_excl, cum_incl)
            const int klo = min(kThreads, max(0, (int)ceil(cum_excl * scale - 0.5)));
            const int khi = min(kThreads, max(0, (int)ceil(cum_incl * scale - 0.5)));
            if (khi > klo) {
              cint[klo] = i | (khi << 16);
              cth[klo] = cum_excl;
            }
          }
          carry += whole;   // (= the last lane's x + before: the next tile's first cum_excl is this tile's last cum_incl)
        }
        __syncthreads();
        {
          // owner of quantile t: the last mark at a position <= t (inclusive max-scan over the 64 positions)
          int pos = (TWK_FIRST64(t) && cint[t] >= 0) ? t : -1;
  #pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, pos, o);
            if (lane >= o) pos = max(pos, y);
          }
          if (lane == 31 && TWK_FIRST64(t)) iscr[1 + warp] = pos;
          __syncthreads();
          if (warp == 1) pos = max(pos, iscr[1]);
          if (!TWK_FIRST64(t)) pos = -1;
          int own = -1;
          double th = 0.0;
          if (pos >= 0) {
            const int mark = cint[pos];
            const int i = mark & 0xffff, khi = mark >> 16;
            if (t < khi) {
              const double cum_excl = cth[pos];
              const double w = raw ? er[i] : fmax(er[i] - avg, 0.0);
              const double th0 = theta[i];
              const double hi = (i + 1 < n) ? theta[i + 1] : kTwoPi;
              const double target = (double(t) + 0.5) / double(kThreads) * W;
              const double frac = (target - cum_excl) * rcp(w);
              th = fma(frac, hi - th0, th0);                           // linear interpolation
              if (!(th > th0 && th < hi)) th = nan("");
              own = i;
            }
          }
          TWK_CHECK(own < 0 || th != th || (th > theta[own] && th < ((own + 1 < n) ? theta[own + 1] : kTwoPi)), 5);
          if (TWK_FIRST64(t)) {
            newth[t] = th;
            newint[t] = own;
          }
        }
        __syncthreads();
        // ---- drop invalid / duplicate angles, compact (ballot + prefix sum) --------------------------------------
        bool v = TWK_FIRST64(t) && (newint[t] >= 0) && (newth[t] == newth[t]);
        if (v && t > 0 && newint[t - 1] == newint[t] && !(newth[t] > newth[t - 1])) v = false;
        const unsigned bal = __ballot_sync(0xffffffffu, v);
        if (lane == 0 && TWK_FIRST64(t)) iscr[1 + warp] = __popc(bal);
        __syncthreads();
        m = iscr[1] + iscr[2];
        const int rank = __popc(bal & ((1u << lane) - 1u)) + (warp ? iscr[1] : 0);
        if (v) {
          cth[rank] = newth[t];
          cint[rank] = newint[t];
        }
        __syncthreads();
        if (m == 0) { exhausted = true; break; }
        // ---- merge: old element j moves up by the number of new samples inserted before it ------------------------
        for (int base = ((n - 1) / TB) * TB; base >= 0; base -= TB) {
          const int j = base + t;
          const bool have = j < n;
          double v0 = 0.0, v1 = 0.0, v2 = 0.0;
          uint16_t v3 = 0;
          int cnt = 0;
          if (have) {
            v0 = theta[j];
            v1 = dA[j];
            v2 = er[j];
            v3 = ids[j];
            int lo = 0, hiq = m;   // cnt = #{r : cint[r] < j}
            while (lo < hiq) {
              const int mid = (lo + hiq) >> 1;
              if (cint[mid] < j) lo = mid + 1; else hiq = mid;
            }
            cnt = lo;
          }
          __syncthreads();
          if (have) {
            theta[j + cnt] = v0;
            dA[j + cnt] = v1;
            er[j + cnt] = v2;
            ids[j + cnt] = v3;
          }
          __syncthreads();
        }
      }   // n > 0
      // ---- solve the new samples (a1-a5 only for the newly added) -----------------------------------------
      const int pos = (t < m) ? cint[t] + 1 + t : 0;
      if (t < m) {
        const double th = cth[t];
        theta[pos] = th;
        ids[pos] = (uint16_t)(n + t);
        double sn, cs;
        if (n == 0) sincospi(double(t) / 32.0, &sn, &cs);   // exactly stage 1's angles
        else sincospi(th * kInvPi, &sn, &cs);               // no range-reduction slow path
        const RecRef in_arena{arena + (size_t)(n + t) * kRecDoubles, 1};
        flags |= point_solve_cs<kScr, kTile>(S.L, S.zc, S.rho, cs, sn, seeds, 1, kTile ? RecRef{tile + t, kThreads} : in_arena,
                                             nullptr, nullptr, nullptr, RecRef{(kTile ? tile : scrbuf) + t, kThreads}, in_arena);
      }
      const int n_new = n + m;
      tile_base = kTile ? n : (1 << 30);
      __syncthreads();
#ifdef TWK_DEBUG
      {   // the sorted list after the merge: angles strictly increasing, ids a permutation of 0 .. n_new - 1
        unsigned* bits = g_twk_stamp + (size_t)blockIdx.x * 128;
        for (int i = t; i < 128; i += TB) bits[i] = 0u;
        __syncthreads();
        for (int i = t; i < n_new; i += TB) {
          TWK_CHECK(i == 0 || theta[i] > theta[i - 1], 1);
          TWK_CHECK(theta[i] >= 0.0 && theta[i] < kTwoPi, 1);
          const unsigned id = ids[i];
          TWK_CHECK(id < (unsigned)n_new, 2);
          if (id < (unsigned)n_new) {
            const unsigned old = atomicOr(&bits[id >> 5], 1u << (id & 31));
            TWK_CHECK(!(old >> (id & 31) & 1u), 2);
          }
        }
        if (t == 0) TWK_DEBUG_COUNT(7);
        __syncthreads();
      }
#endif
      // ---- re-evaluate only the intervals that changed: the one to the left of every new sample, and the
      //      one to its right when the next sample is old (or the list wraps around) ---------------------------------
      int viol = 0;
      if (t < m) {
        const bool last_in_group = (t == m - 1) || (cint[t + 1] != cint[t]);
#pragma unroll 1
        for (int side = 0; side < 2; ++side) {
          if (side == 0 ? (pos == 0) : !last_in_group) continue;
          const int ia = pos - 1 + side;                       // interval (ia, ia + 1)
          const int ib = (ia + 1 < n_new) ? ia + 1 : 0;
          const double dth = (ia + 1 < n_new) ? theta[ia + 1] - theta[ia] : kTwoPi - theta[ia];
          Piece P = eval_interval(recref(ids[ia]), recref(ids[ib]), dth, p.slope_gate2, p.slope_cos2);
          if (kGuard && P.crossing == 0 && n_new >= 4) P.err += guard_term(ia, n_new);
          dA[ia] = P.dA;
          er[ia] = P.err;
          viol |= P.slope;
        }
      }
      n = n_new;
      // ---- a5, slope detector: a crossing whose real pair is not perpendicular to the neighbouring ghost
      //      pair is re-judged.  Rare: out-of-line repair rounds over ALL intervals until none is flagged.  Each round:
      //      evaluate everything, list the flagged crossings, re-judge the pairs flagged by a creation (the record to
      //      the right of the interval), then those flagged by an annihilation (the record to the left, if it still has
      //      five images). ------------------------------------------------------------------------------------------
      if (__syncthreads_or(viol)) {
        slope_seen = true;
        tile_base = 1 << 30;   // the repair rounds change records: from here on only the arena's copies are used
        for (int round = 0; round < 4096; ++round) {
          if (t == 0) iscr[3] = 0;
          __syncthreads();
          for (int i = t; i < n; i += TB) {
            const int ib = (i + 1 < n) ? i + 1 : 0;
            const double dth = (i + 1 < n) ? theta[i + 1] - theta[i] : kTwoPi - theta[i];
            Piece P = eval_interval_cold(recref(ids[i]), recref(ids[ib]), dth, p.slope_gate2, p.slope_cos2);
            if (kGuard && P.crossing == 0 && n >= 4) P.err += guard_term(i, n);
            dA[i] = P.dA;
            er[i] = P.err;
            if (P.slope) {
              const int k = atomicAdd(&iscr[3], 1);
              if (k < kThreads) {
                newint[k] = i;
                cint[k] = (P.slope & 255) | (P.crossing > 0 ? 256 : 0);
              }
            }
          }
          __syncthreads();
          const int nv = min(iscr[3], kThreads);
          if (nv == 0) break;
#ifdef TWK_DEBUG
          unsigned* bits = g_twk_stamp + (size_t)blockIdx.x * 128;     // one writer per record per phase
          for (int i = t; i < 128; i += TB) bits[i] = 0u;
          __syncthreads();
#endif
          if (t < nv && (cint[t] & 256)) {
            const int ib = (newint[t] + 1 < n) ? newint[t] + 1 : 0;
#ifdef TWK_DEBUG
            TWK_CHECK(!(atomicOr(&bits[ids[ib] >> 5], 1u << (ids[ib] & 31)) >> (ids[ib] & 31) & 1u), 3);
#endif
            demote_pair(recref(ids[ib]), cint[t] & 15, (cint[t] >> 4) & 15);
          }
          __syncthreads();
#ifdef TWK_DEBUG
          for (int i = t; i < 128; i += TB) bits[i] = 0u;
          __syncthreads();
#endif
          if (t < nv && !(cint[t] & 256)) {
            const RecRef S5 = recref(ids[newint[t]]);
#ifdef TWK_DEBUG
            const unsigned idw = ids[newint[t]];
            TWK_CHECK(!(atomicOr(&bits[idw >> 5], 1u << (idw & 31)) >> (idw & 31) & 1u), 3);
#endif
            if (S5.nreal() == 5) demote_pair(S5, cint[t] & 15, (cint[t] >> 4) & 15);
          }
          __syncthreads();
        }
      }
    }

    // ---- outputs / hand-over ------------------------------------------------------------------------------------
    const int rep = __syncthreads_or(flags & kPointRepaired);
    const int nonf = __syncthreads_or(flags & (kPointNonFinite | kPointGuard));
    const int slp = __syncthreads_or(flags & kPointSlope);
    if (t == 0) {
      iscr[0] = next_cur;   // (every thread read the current entry before the barriers above)
      if (exhausted && !p.final_stage) {
        const int slot = atomicAdd(p.next_count, 1);
        TWK_CHECK(slot >= 0 && slot < p.b.n_sources, 4);
        p.next_list[slot] = (int32_t)src;
        if (kTile) iscr[5] = slot;
      } else {
        if (exhausted) status |= 2u;
        if (rep) status |= 4u;
        if (nonf) status |= 16u;
        if (slope_seen || slp) status |= 32u;
        p.out_mu[src] = A * rcp(kPi * S.rho * S.rho);
        if (p.out_err) p.out_err[src] = E * rcp(fabs(A));
        if (p.out_nsamples) p.out_nsamples[src] = n;
        if (p.out_status) p.out_status[src] = status;
      }
    }
    if (kTile && exhausted && !p.final_stage && p.carry_role == 1) {   // (uniform) the state goes along to the next stage
      __syncthreads();
      const long long slot = iscr[5];
      if (slot < p.carry_slots && n <= p.carry_cap)
        carry_out(p.carry + (size_t)slot * carry_doubles(p.carry_cap), p.carry_cap, n, theta, dA, er, ids, arena, hand,
                  (int)((status & ~S.status) | (rep ? 4u : 0u) | (nonf ? 16u : 0u) | ((slope_seen || slp) ? 32u : 0u)));
    }
  }
}

#undef TWK_FIRST64

}  // namespace twk
