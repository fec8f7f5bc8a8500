// twk_refine1.cuh -- stage 1.5 of twk_magnify: the FIRST refinement iteration (64 -> up to 128 samples) of the
// sources stage 1 handed over, entirely in shared memory.
//
// Most sources that need refinement at all need exactly this one iteration (88 % of BASELINE config 3's, DESIGN.md
// section 5), and for it everything is small and known in advance: the 64 old records come from the hand-over slot (copied
// asynchronously into a [26][64] tile while the sampler runs), the <= 64 new records go to a second tile, the sorted
// state is at most 128 entries, the weight scan is a single tile.  The arithmetic is, operation for operation, that of
// adaptive_kernel's iteration on the same inputs (same sums, same scan, same quantile rule, same point solve, same
// interval evaluation): a source that converges here gets the value stage 2 would have given it.  A source that does
// NOT converge here (or whose slope detector fires, or that produced no valid new angle) is left untouched: its entry
// goes on the worklist of stage 2, which starts from the hand-over slot as before.  Entries without a hand-over slot are
// passed on unchanged.
#pragma once

#include "twk_adaptive.cuh"

namespace twk {

struct Refine1Args {
  Batch b;
  double tol;
  double slope_gate2, slope_cos2;
  int subtract_avg_tol;
  const int32_t* list;     // stage 1's worklist (source ids), entry e
  const int* count;        // its length (device)
  int* cursor;             // work fetch counter (zeroed before launch)
  const double* handoff;   // hand-over arena: entry e < handoff_slots has slot e
  long long handoff_slots;
  int32_t* next_list;      // OUT: entries (indices into `list` / the hand-over arena) that stage 2 still has to refine
  int* next_count;
  double* out_mu;
  double* out_err;         // may be null
  int32_t* out_nsamples;   // may be null
  uint32_t* out_status;    // may be null
};

constexpr int kR1Cap = 2 * kThreads;   // 128 sorted entries at most
constexpr int kR1Chunk = 8;            // worklist entries per work fetch, at most

__host__ __device__ constexpr size_t refine1_smem_bytes() {
  // tiles A, B [26][64] | theta, dA, er [128] | newth, cth [64] | scratch [8] | seeds [32] | newint, cint [64] | iscr [8] | ids [128]
  return (size_t)(2 * kRecDoubles * kThreads + 3 * kR1Cap + 2 * kThreads + 8 + 32) * 8 + (size_t)(2 * kThreads + 8) * 4 +
         (size_t)kR1Cap * 2;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

__global__ void __launch_bounds__(kThreads, 6) refine1_kernel(Refine1Args p) {
  extern __shared__ double sm[];
  double* tileA = sm;                               // [26][64] records 0..63 (copy of the hand-over slot's)
  double* tileB = tileA + kRecDoubles * kThreads;   // [26][64] records 64.. (this iteration's new samples)
  double* theta = tileB + kRecDoubles * kThreads;   // [128] sorted sample angles
  double* dA = theta + kR1Cap;                      // [128] area piece of interval (i, i+1)
  double* er = dA + kR1Cap;                         // [128] error piece of interval (i, i+1)
  double* newth = er + kR1Cap;                      // [64] angle of quantile k
  double* cth = newth + kThreads;                   // [64] compacted new angles
  double* scratch = cth + kThreads;                 // [8]
  double* seeds = scratch + 8;                      // [31 (+1)]
  int* newint = reinterpret_cast<int*>(seeds + 32); // [64] interval of quantile k
  int* cint = newint + kThreads;                    // [64] compacted
  int* iscr = cint + kThreads;                      // [8]: -, two warp counts, -, chunk, entries of the chunk to do
  uint16_t* ids = reinterpret_cast<uint16_t*>(iscr + 8);   // [128] record id of the sample at each sorted position

  const int t = threadIdx.x;
  const int lane = t & 31, warp = t >> 5;
  auto recref = [&](int id) -> RecRef {
    return (id < kThreads) ? RecRef{tileA + id, kThreads} : RecRef{tileB + (id - kThreads), kThreads};
  };
  const long long total = (long long)*p.count;
  constexpr int n = kThreads;   // samples on entry: the 64 of the first iteration

  // Work comes in chunks of kR1Chunk entries.  Entries that are not for this stage -- no hand-over slot (stage 2 recomputes
  // such a source from its first sample), or marked by stage 1 as a source whose error is spread too evenly for one
  // iteration to finish it -- are passed on at once, all of the chunk's with one atomic (a batch in which nothing is for
  // this stage, BASELINE config 5, costs one list read per entry); the others are taken one after the other.
  // (a short worklist goes out entry by entry, so that every CTA gets some)
  const int kc = (int)max(1LL, min((long long)kR1Chunk, total / ((long long)gridDim.x * 4)));
  for (;;) {
    __syncthreads();
    if (t == 0) iscr[4] = atomicAdd(p.cursor, kc);
    __syncthreads();
    const long long chunk = iscr[4];
    if (chunk >= total) break;
    if (warp == 0) {
      const long long e = chunk + lane;
      const bool valid = lane < kc && e < total;
      const bool skip = valid && (e >= p.handoff_slots || p.list[e] < 0);
      const unsigned skips = __ballot_sync(0xffffffffu, skip), valids = __ballot_sync(0xffffffffu, valid);
      int off = 0;
      if (lane == 0 && skips) off = atomicAdd(p.next_count, __popc(skips));
      off = __shfl_sync(0xffffffffu, off, 0);
      if (skip) p.next_list[off + __popc(skips & ((1u << lane) - 1u))] = (int32_t)e;
      if (lane == 0) iscr[5] = (int)(valids & ~skips);
#ifdef TWK_DEBUG
      if (skip) TWK_DEBUG_COUNT(11);
      if (skip) TWK_CHECK(off + __popc(skips & ((1u << lane) - 1u)) < total, 4);
#endif
    }
    __syncthreads();
    const unsigned todo = (unsigned)iscr[5];
#pragma unroll 1
    for (int b = 0; b < kc; ++b) {
    if (!(todo >> b & 1u)) continue;
    const long long cur = chunk + b;
    bool pass_on = false;   // (uniform) leave this entry to stage 2 after all
    const double* hand = p.handoff + (size_t)cur * kHandDoubles;
    TWK_CHECK(cur >= 0 && cur < total && cur < p.handoff_slots, 4);
    if (t == 0) TWK_DEBUG_COUNT(8);
    long long src = 0;
    SourceParams S;
    S.valid = false;
    int flags = 0;
    double A = 0.0, E = 0.0;
    int m = 0, n_new = n;
    if (!pass_on) {
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
      theta[t] = kTwoPi * double(t) / double(kThreads);
      ids[t] = (uint16_t)t;
      dA[t] = hand[kRecDoubles * kThreads + t];
      er[t] = hand[(kRecDoubles + 1) * kThreads + t];
      if (t < kSeedDoubles) seeds[t] = hand[(kRecDoubles + 2) * kThreads + t];
      flags |= code_of(hand[kNR * kThreads + t]) >> 3;   // point flags of the old records (row 25 of the slot)
      __syncthreads();
      // ---- sums over the 64 intervals (as adaptive_kernel: strided partial sums, block tree) ---------------------------
      double a = dA[t], e = er[t];
      block_sum2(a, e, scratch);
      A = a;
      E = e;
      const double tolA = p.tol * fabs(A);
      // (stage 1 found this source unfinished from the same sums; the tests are kept for the degenerate cases)
      if (!(isfinite(A) && isfinite(E)) || E <= tolA) pass_on = true;
      if (!pass_on) {
        // ---- a8: error-weighted inverse-transform sampling, 64 quantiles, one tile ------------------------
        const double avg = p.subtract_avg_tol ? tolA / double(n) : 0.0;   // "average tolerance", reading A-5
        double W = fmax(er[t] - avg, 0.0), unused = 0.0;
        block_sum2(W, unused, scratch);
        const bool raw = !(W > 0.0);
        if (raw) W = E;
        const double scale = double(kThreads) / W;
        cint[t] = -1;
        int kq = 0;   // quantiles (new samples) this thread's interval gets
        __syncthreads();
        {
          const int i = t;
          const double w = raw ? er[i] : fmax(er[i] - avg, 0.0);
          double x = w;   // inclusive scan over the 64 threads
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const double y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += y;
          }
          __syncthreads();
          if (lane == 31) scratch[4 + warp] = x;
          __syncthreads();
          const double w0 = scratch[4];
          double before = 0.0;
          if (warp == 1) before = w0;
          const double carry = 0.0;
          const double cum_incl = carry + (x + before);
          double cum_excl = __shfl_up_sync(0xffffffffu, cum_incl, 1);
          if (lane == 0) cum_excl = carry + before;
          if (w > 0.0) {
            const int klo = min(kThreads, max(0, (int)ceil(cum_excl * scale - 0.5)));
            const int khi = min(kThreads, max(0, (int)ceil(cum_incl * scale - 0.5)));
            if (khi > klo) {
              cint[klo] = i | (khi << 16);
              cth[klo] = cum_excl;
              kq = khi - klo;
            }
          }
        }
        // Will these quantiles do?  Interval i gets k_i new samples; with its error falling like the square of the
        // refinement, the sum after this iteration would be about sum e_i / (k_i + 1)^2.  Above the tolerance: not worth
        // trying here (calibrated on the oracle over BASELINE configs 3-5 and the Fig.5 maps: 92-98 % of the sources that
        // pass converge in this iteration, 1 % of those that would have converged are turned away); stage 2 takes it.
        {
          const double kk = double(kq + 1);
          double pr = er[t] * rcp(kk * kk), unused2 = 0.0;
          block_sum2(pr, unused2, scratch);   // (its barriers also publish the marks in cint / cth)
          if (pr > tolA) pass_on = true;
        }
        if (!pass_on) {   // (still inside the sampler's scope: avg, raw, W)
        // the 64 records: 832 16-byte chunks, 13 per thread, straight from the slot into tile A; not waited for before
        // the interval evaluations need them
        {
          const char* g = reinterpret_cast<const char*>(hand);
          char* s = reinterpret_cast<char*>(tileA);
#pragma unroll
          for (int k = 0; k < (kRecDoubles * kThreads * 8) / (16 * kThreads); ++k) cp_async16(s + (k * kThreads + t) * 16, g + (k * kThreads + t) * 16);
          cp_async_commit();
        }
        {
          // owner of quantile t: the last mark at a position <= t (inclusive max-scan over the 64 positions)
          int pos = (cint[t] >= 0) ? t : -1;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, pos, o);
            if (lane >= o) pos = max(pos, y);
          }
          if (lane == 31) iscr[1 + warp] = pos;
          __syncthreads();
          if (warp == 1) pos = max(pos, iscr[1]);
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
          newth[t] = th;
          newint[t] = own;
        }
        __syncthreads();
        // ---- drop invalid / duplicate angles, compact (ballot + prefix sum) ------------------------------------------
        bool v = (newint[t] >= 0) && (newth[t] == newth[t]);
        if (v && t > 0 && newint[t - 1] == newint[t] && !(newth[t] > newth[t - 1])) v = false;
        const unsigned bal = __ballot_sync(0xffffffffu, v);
        if (lane == 0) iscr[1 + warp] = __popc(bal);
        __syncthreads();
        m = iscr[1] + iscr[2];
        const int rank = __popc(bal & ((1u << lane) - 1u)) + (warp ? iscr[1] : 0);
        if (v) {
          cth[rank] = newth[t];
          cint[rank] = newint[t];
        }
        __syncthreads();
        if (m == 0) pass_on = true;   // (stage 2 comes to the same conclusion and sends the source on)
#ifdef TWK_DEBUG
        if (t < m) {   // a new angle lies strictly inside the interval that owns its quantile; owners do not decrease
          const int i = cint[t];
          TWK_CHECK(i >= 0 && i < n && cth[t] > theta[i] && cth[t] < ((i + 1 < n) ? theta[i + 1] : kTwoPi), 5);
          TWK_CHECK(t == 0 || cint[t - 1] <= i, 5);
        }
#endif
        }
      }
    }
    int viol = 0;
    if (!pass_on) {
      // ---- merge: old element j moves up by the number of new samples inserted before it (one tile) -----------------
      {
        const int j = t;
        const double v0 = theta[j], v1 = dA[j], v2 = er[j];
        const uint16_t v3 = ids[j];
        int lo = 0, hiq = m;   // cnt = #{r : cint[r] < j}
        while (lo < hiq) {
          const int mid = (lo + hiq) >> 1;
          if (cint[mid] < j) lo = mid + 1; else hiq = mid;
        }
        const int cnt = lo;
        __syncthreads();
        theta[j + cnt] = v0;
        dA[j + cnt] = v1;
        er[j + cnt] = v2;
        ids[j + cnt] = v3;
        __syncthreads();
      }
      // ---- solve the new samples (a1-a5) into tile B ---------------------------------------------------------------------
      const int pos = (t < m) ? cint[t] + 1 + t : 0;
      if (t < m) {
        const double th = cth[t];
        theta[pos] = th;
        ids[pos] = (uint16_t)(n + t);
        double sn, cs;
        sincospi(th * kInvPi, &sn, &cs);
        const RecRef rec{tileB + t, kThreads};
        flags |= point_solve_cs<true, false>(S.L, S.zc, S.rho, cs, sn, seeds, 1, rec, nullptr, nullptr, nullptr, rec);
      }
      n_new = n + m;
      cp_async_wait_all();   // this thread's chunks of tile A have landed ...
      __syncthreads();       // ... and so have everybody else's; the new records are complete
#ifdef TWK_DEBUG
      for (int i = t; i < n_new; i += kThreads) {
        TWK_CHECK(ids[i] < n_new, 0);
        if (i + 1 < n_new) TWK_CHECK(theta[i] < theta[i + 1], 1);
        int seen = 0;   // record id i sits at exactly one sorted position
        for (int j = 0; j < n_new; ++j) seen += (ids[j] == i);
        TWK_CHECK(seen == 1, 2);
      }
      if (t == 0) {
        TWK_DEBUG_COUNT(6);
        TWK_DEBUG_COUNT(7);
        TWK_DEBUG_COUNT(9);
      }
#endif
      // ---- re-evaluate only the intervals that changed ------------------------------------------------------------
      if (t < m) {
        const bool last_in_group = (t == m - 1) || (cint[t + 1] != cint[t]);
#pragma unroll 1
        for (int side = 0; side < 2; ++side) {
          if (side == 0 ? (pos == 0) : !last_in_group) continue;
          const int ia = pos - 1 + side;                       // interval (ia, ia + 1)
          const int ib = (ia + 1 < n_new) ? ia + 1 : 0;
          const double dth = (ia + 1 < n_new) ? theta[ia + 1] - theta[ia] : kTwoPi - theta[ia];
          const Piece P = eval_interval(recref(ids[ia]), recref(ids[ib]), dth, p.slope_gate2, p.slope_cos2);
          dA[ia] = P.dA;
          er[ia] = P.err;
          viol |= P.slope;
        }
      }
      // a5, slope detector: a flagged crossing needs the repair rounds of adaptive_kernel -- rare; such a source is left to
      // stage 2 (which starts again from the hand-over slot)
      if (__syncthreads_or(viol)) pass_on = true;
    } else {
      cp_async_wait_all();   // (nothing of this entry may still be in flight when the tile is reused)
    }
    bool finished = false;
    if (!pass_on) {
      // ---- sums over the n_new intervals and the stop rule -------------------------------------------------------
      double a = 0.0, e = 0.0;
      for (int i = t; i < n_new; i += kThreads) {
        a += dA[i];
        e += er[i];
      }
      block_sum2(a, e, scratch);
      A = a;
      E = e;
      finished = isfinite(A) && isfinite(E) && E <= p.tol * fabs(A);
    }
    const int rep = __syncthreads_or(flags & kPointRepaired);
    const int nonf = __syncthreads_or(flags & (kPointNonFinite | kPointGuard));
    const int slp = __syncthreads_or(flags & kPointSlope);
    if (t == 0) {
      if (finished) {
        uint32_t status = S.status | 1u;
        if (rep) status |= 4u;
        if (nonf) status |= 16u;
        if (slp) status |= 32u;
        p.out_mu[src] = A * rcp(kPi * S.rho * S.rho);
        if (p.out_err) p.out_err[src] = E * rcp(fabs(A));
        if (p.out_nsamples) p.out_nsamples[src] = n_new;
        if (p.out_status) p.out_status[src] = status;
        TWK_DEBUG_COUNT(10);
      } else {
        const int at = atomicAdd(p.next_count, 1);
        TWK_CHECK(at >= 0 && at < total, 4);
        p.next_list[at] = (int32_t)cur;   // stage 2 takes it from its hand-over slot
      }
    }
    }   // entries of the chunk
  }
}

}  // namespace twk
