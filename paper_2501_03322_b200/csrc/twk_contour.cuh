// twk_contour.cuh -- per-sample record (a1, a4, a5) and per-interval link + area + error (a6, a7).
// See twk_device.cuh for the citation key.
#pragma once

#include <string.h>

#include "twk_device.cuh"

namespace twk {

// ------------------------------------------------------------------------------------------------------------
// Sample record: what an interval needs from one boundary sample.  26 doubles, element e at base[e * stride]:
//   [0..4]  Re z      slots 0,1 = positive-parity images, slots 2,3,4 = negative-parity images
//   [5..9]  Im z      (a sample with 3 real images keeps its GHOST pair's positions in the z fields of slots 1 and 4:
//                     the slope detector compares directions across a count change)
//   [10..14] Re z'    z' = dz/dtheta, Eq.(10) (conj on f' restored)
//   [15..19] Im z'
//   [20..24] z'^z''   Eq.(10) (division by J restored)
//   [25]    nreal (3 or 5) + 8 * point flags (kPoint*), an integer kept as raw bits
// In shared memory the record is a column of a [26][TILE] array (stride = TILE, conflict-free); in the global
// arena it is 26 contiguous doubles (stride = 1, 208 B).
// ------------------------------------------------------------------------------------------------------------
constexpr int kRecDoubles = 26;
constexpr int kZX = 0, kZY = 5, kPX = 10, kPY = 15, kW = 20, kNR = 25;

TWK_HD int code_of(double d) {
#ifdef __CUDA_ARCH__
  return (int)__double_as_longlong(d);
#else
  long long v;
  memcpy(&v, &d, 8);
  return (int)v;
#endif
}
TWK_HD double code_as_double(int c) {
#ifdef __CUDA_ARCH__
  return __longlong_as_double((long long)c);
#else
  long long v = c;
  double d;
  memcpy(&d, &v, 8);
  return d;
#endif
}

struct RecRef {
  double* base;
  int stride;
  TWK_HD double& at(int e) const { return base[e * stride]; }
  TWK_HD cd z(int slot) const { return mk(base[(kZX + slot) * stride], base[(kZY + slot) * stride]); }
  TWK_HD cd zp(int slot) const { return mk(base[(kPX + slot) * stride], base[(kPY + slot) * stride]); }
  TWK_HD double w(int slot) const { return base[(kW + slot) * stride]; }
  // element kNR holds an integer code as raw bits (no int <-> double conversion on the hot path)
  TWK_HD int code() const { return code_of(base[kNR * stride]); }
  TWK_HD int nreal() const { return code() & 7; }
  TWK_HD int point_flags() const { return code() >> 3; }
  TWK_HD void set_code(int c) const { base[kNR * stride] = code_as_double(c); }
};

constexpr int kPointRepaired = 1;   // parity sum was not -1 and was repaired (G-5)
constexpr int kPointSlope = 4;      // a real pair was re-judged as ghosts by the slope detector
constexpr int kPointNonFinite = 2;  // a root or a derived quantity is not finite
constexpr int kPointGuard = 8;      // the sample sat on a lens and was moved off it (reading B-1)
constexpr int kPointRecovered = 16; // diagnostics: the seeded solve went through its Vieta recovery
constexpr int kPointCold = 32;      // diagnostics: the cold solver was used (no seeds, or the seeded solve failed)

// B-1: a boundary point ON a lens (conj(y) = 0 or conj(y) = -s) makes c5 = 0: one root escapes to infinity
// and one sits on the pole of f.  The magnification is continuous there, so a point closer to a lens than 1e-14 s --
// the rounding of zeta itself -- is moved to that distance along the lens axis.  Returns true when it fired.
TWK_HD bool lens_guard(cd& y, double s) {
  const double dmin = 1e-14 * s;
  bool fired = false;
  if (norm2(y) < dmin * dmin) { y = mk(dmin, 0.0); fired = true; }
  if (norm2(mk(y.x + s, y.y)) < dmin * dmin) { y = mk(-s + dmin, 0.0); fired = true; }
  return fired;
}

// ------------------------------------------------------------------------------------------------------------
// a1 + a2 + a3 + a4 + a5: one boundary point source.
// Writes the record; optionally the five roots (CM frame), their kinds and the real-image count.
// ------------------------------------------------------------------------------------------------------------
// cs, sn = cos(theta), sin(theta).  seeds: nullptr = cold solve; otherwise the source's seed block written by
// centre_seeds() (element e at seeds[e * seed_stride]): every root of the boundary sample is predicted to first order
// from the centre's root, eta_k + A_k delta + B_k conj(delta) with delta = rho e^{i theta}, and refined by the seeded
// Newton solve, with the cold solver as verified fallback.
// kScr: `scr` is per-thread scratch of >= 20 elements in SHARED memory (it may be the record itself: the scratch is dead
// before the record is written).  The residual detector then parks the roots and their residuals there and fetches the
// two largest-|R| ones by index: 28 shared-memory accesses instead of ~140 register selects.
// kDual: the record is also written to `rec2` (the refinement kernel keeps a shared-memory copy of the new records
// next to the arena's).
template <bool kScr = false, bool kDual = false>
TWK_HD int point_solve_cs(const Lens& L, cd zc, double rho, double cs, double sn, const double* seeds, int seed_stride,
                          RecRef rec, double* out_z, int8_t* out_kind, int8_t* out_count, RecRef scr = RecRef{nullptr, 0},
                          RecRef rec2 = RecRef{nullptr, 0}) {
  const cd zeta = mk(fma(rho, cs, zc.x), fma(rho, sn, zc.y));
  const cd dzeta = mk(-rho * sn, rho * cs);                     // zeta' = i rho e^{i theta}
  cd y = mk(zeta.x - L.z2, zeta.y);
  cd c[6], eta[5];
  coeffs_eq6(y, L.s, L.m2, c);
  // next to a lens (closer than ~1e-8 s) one root runs off towards infinity and one onto the pole: such a sample is left
  // to the cold solver; ON the lens it is moved off it first (B-1).  |c5| = |y| |y + s| measures the distance to the
  // nearer lens (the other factor is within [s/2, ...]): |c5| < 1e-8 s^2 <=> closer than (1..2) 1e-8 s
  const double n5 = norm2(c[5]), s2 = L.s * L.s;
  const bool near_lens = !(n5 >= 1e-16 * (s2 * s2));
  bool guarded = false;
  if (near_lens) {
    guarded = lens_guard(y, L.s);
    if (guarded) {
      const Coef6 C = coeffs_eq6_cold(y, L.s, L.m2);
#pragma unroll
      for (int i = 0; i < 6; ++i) c[i] = C.c[i];
    }
  }
  int solved = 0;
  if (seeds && !near_lens) {
    const double dx = rho * cs, dy = rho * sn;                  // delta
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      const double ex = seeds[k * seed_stride], ey = seeds[(5 + k) * seed_stride];
      const double pxx = seeds[(10 + k) * seed_stride], pxy = seeds[(15 + k) * seed_stride];
      const double pyx = seeds[(20 + k) * seed_stride], pyy = seeds[(25 + k) * seed_stride];
      // eta + A delta + B conj(delta) as a real 2 x 2 map of (Re delta, Im delta), prepared by centre_seeds()
      eta[k] = mk(fma(pxx, dx, fma(pxy, dy, ex)), fma(pyx, dx, fma(pyy, dy, ey)));
    }
    {   // the seeded solve works on the monic quintic; the cold solver below gets the same coefficients with c5 = 1
      const double r5 = rcp(n5);
      const cd i5 = mk(c[5].x * r5, -c[5].y * r5);
#pragma unroll
      for (int i = 0; i < 5; ++i) c[i] = c[i] * i5;
      c[5] = mk(1.0, 0.0);
    }
    solved = quintic_roots_seeded(c, eta, seeds[30 * seed_stride] != 0.0);
  }
  int flags = (guarded ? kPointGuard : 0) | (solved == 2 ? kPointRecovered : 0) | (solved ? 0 : kPointCold);
  if (!solved) {
    TWK_COUNT(cold_solve);
    Coef6 C;
#pragma unroll
    for (int i = 0; i < 6; ++i) C.c[i] = c[i];
    const Roots5 R = quintic_roots_cold(C);
#pragma unroll
    for (int k = 0; k < 5; ++k) eta[k] = R.r[k];
  }

  // a4: f', f'', residual, Jacobian in the planet frame (z2 - z = -eta, z1 - z = -s - eta; both are frame
  // invariant)
  cd fp[5], a3[5], b3[5], Res[5];
  double J[5], R2[5];
  bool finite = true;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    // a = 1 / (z1 - z), b = 1 / (z2 - z): ONE reciprocal for both, 1 / (|z1 - z|^2 |z2 - z|^2)
    const cd za = mk(-L.s - eta[k].x, -eta[k].y), zb = -eta[k];
    const double na = norm2(za), nb = norm2(zb);
    const double rab = rcp(na * nb);
    const double ia_ = rab * nb, ib_ = rab * na;
    const cd a = mk(za.x * ia_, -za.y * ia_), b = mk(zb.x * ib_, -zb.y * ib_);
    const cd a2 = a * a, b2 = b * b;
    fp[k] = L.m1 * a2 + L.m2 * b2;                       // Eq.(7)
    a3[k] = a2 * a;                                      // f'' is finished below, for the real images only
    b3[k] = b2 * b;
    // Eq.(12): R = y - eta - conj(f), f = m1 a + m2 b folded into the subtraction
    Res[k] = mk(fma(-L.m1, a.x, fma(-L.m2, b.x, y.x - eta[k].x)), fma(L.m1, a.y, fma(L.m2, b.y, y.y - eta[k].y)));
    J[k] = fma(-fp[k].x, fp[k].x, fma(-fp[k].y, fp[k].y, 1.0));   // Eq.(7): 1 - |f'|^2
    R2[k] = norm2(Res[k]);
  }
  {   // all ten finite?  |R|^2 >= 0 and J <= 1: their sums cannot cancel an infinity and NaN propagates
    const double sr = ((R2[0] + R2[1]) + (R2[2] + R2[3])) + R2[4], sj = ((J[0] + J[1]) + (J[2] + J[3])) + J[4];
    finite = isfinite(sr) && isfinite(sj);
  }
  // a5: residual detector, 2-cycle reading (G-1): the two largest-|R| roots (ia, ib) are a ghost pair iff
  // R_ia = eta_ib - eta_ia and R_ib = eta_ia - eta_ib ("a pair of ghost images with opposite residuals").
  // (running maxima in scalars: no dynamically indexed array, everything stays in registers)
  int ia = 0, ib = -1;
  double mA = R2[0], mB = -1.0;
  cd eA = eta[0], rA = Res[0], eB = eta[0], rB = Res[0];
  if (kScr) {
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      scr.at(k) = eta[k].x;
      scr.at(5 + k) = eta[k].y;
      scr.at(10 + k) = Res[k].x;
      scr.at(15 + k) = Res[k].y;
    }
    // the two largest |R|^2 by integer maxima over keys (high word of the non-negative double, index in the low three
    // bits): |R|^2 of a ghost is orders of magnitude above the rounding residue of a real image, 2^-17 relative resolves
    // every case that matters; among real images (or between the two ghosts, whose |R| are equal) any order will do
    unsigned key[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) key[k] = ((unsigned)__double2hiint(R2[k]) & ~7u) | (unsigned)k;
    const unsigned t1 = max(key[0], key[1]), s1 = min(key[0], key[1]), t2 = max(key[2], key[3]), s2 = min(key[2], key[3]);
    const unsigned T4 = max(t1, t2), U4 = max(min(t1, t2), max(s1, s2));   // first and second of the first four
    const unsigned T5 = max(T4, key[4]), U5 = max(min(T4, key[4]), U4);
    ia = (int)(T5 & 7u);
    const int jb = (int)(U5 & 7u);
    ib = jb;
    eA = mk(scr.at(ia), scr.at(5 + ia));
    rA = mk(scr.at(10 + ia), scr.at(15 + ia));
    eB = mk(scr.at(jb), scr.at(5 + jb));
    rB = mk(scr.at(10 + jb), scr.at(15 + jb));
    mA = norm2(rA);   // (= R2[ia], R2[ib] bit for bit)
    mB = norm2(rB);
  } else {
#pragma unroll
    for (int k = 1; k < 5; ++k) {
      if (R2[k] > mA) {          // new largest: the old largest becomes the second
        mB = mA; ib = ia; eB = eA; rB = rA;
        mA = R2[k]; ia = k; eA = eta[k]; rA = Res[k];
      } else if (R2[k] > mB) {
        mB = R2[k]; ib = k; eB = eta[k]; rB = Res[k];
      }
    }
  }
  const cd dab = eB - eA;
  const bool ghost = norm2(rA - dab) < mA && norm2(rB + dab) < mB;
  // kinds as bit masks over the five roots: gmask = ghost pair, posm / negm = real images of positive / negative parity
  // (Eq.(7): p = sign J)
  const unsigned gmask = ghost ? ((1u << ia) | (1u << (ib & 7))) : 0u;
  unsigned jpos = 0;
#pragma unroll
  for (int k = 0; k < 5; ++k) jpos |= (J[k] > 0.0) ? (1u << k) : 0u;
  unsigned posm = jpos & ~gmask, negm = ~jpos & ~gmask & 31u;
  const int nreal = 5 - __popc(gmask);
  int npos = __popc(posm);
  // parity sum must be -1.  Repair by flipping the smallest-|J| image of the over-represented parity.
  flags |= finite ? 0 : kPointNonFinite;
  const int want = (nreal - 1) >> 1;
  for (int guard = 0; guard < 5 && npos != want; ++guard) {
    const bool over = npos > want;
    const unsigned cand = over ? posm : negm;
    int best = -1;
    double bj = 1e300;
#pragma unroll
    for (int k = 0; k < 5; ++k)
      if ((cand >> k & 1u) && fabs(J[k]) < bj) { bj = fabs(J[k]); best = k; }
    if (best >= 0) {
      posm ^= 1u << best;
      negm ^= 1u << best;
    }
    npos += over ? -1 : 1;
    flags |= kPointRepaired;
  }
  // record: positives to slots 0.., negatives to slots 2..: the slot of a root is the number of same-parity roots before it
  int sp = 0, sm = 2;
  const double m1x2 = L.m1 + L.m1, m2x2 = L.m2 + L.m2, rho2 = rho * rho;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const cd z = mk(eta[k].x + L.z2, eta[k].y);
    const bool isp = posm >> k & 1u, isn = negm >> k & 1u;
    if (out_z) { out_z[2 * k] = z.x; out_z[2 * k + 1] = z.y; }
    if (out_kind) out_kind[k] = (int8_t)(isp ? 1 : (isn ? -1 : 0));
    const int slot = isp ? sp : sm;   // = the number of same-parity roots before this one (+ 2 for the negatives)
    sp += isp ? 1 : 0;
    sm += isn ? 1 : 0;
    // (slots stay inside the record whatever the kinds are: with non-finite J every root counts as negative)
    if ((isp || isn) && slot < (isp ? 2 : 5)) {
      const double invJ = rcp1(J[k]);   // (40 bits: z' and z'^z'' only enter the parabolic corrections and the estimates)
      // z' = (zeta' - conj(f') conj(zeta')) / J                       Eq.(10), repaired (E-2)
      // (conj(f') conj(zeta') = conj(f' zeta'), folded into the subtraction)
      const cd zp = mk(fma(fp[k].y, dzeta.y, fma(-fp[k].x, dzeta.x, dzeta.x)) * invJ,
                       fma(fp[k].x, dzeta.y, fma(fp[k].y, dzeta.x, dzeta.y)) * invJ);
      // z'^z'' = (rho^2 + Im[z'^2 zeta' f'']) / J                     Eq.(10), repaired (E-3);  f'' = 2 (m1 a^3 + m2 b^3)
      const cd fpp = mk(fma(m1x2, a3[k].x, m2x2 * b3[k].x), fma(m1x2, a3[k].y, m2x2 * b3[k].y));
      const cd zp2 = zp * zp, zf = dzeta * fpp;
      const double w = fma(zp2.x, zf.y, fma(zp2.y, zf.x, rho2)) * invJ;
      rec.at(kZX + slot) = z.x;
      rec.at(kZY + slot) = z.y;
      rec.at(kPX + slot) = zp.x;
      rec.at(kPY + slot) = zp.y;
      rec.at(kW + slot) = w;
      if (kDual) {
        rec2.at(kZX + slot) = z.x;
        rec2.at(kZY + slot) = z.y;
        rec2.at(kPX + slot) = zp.x;
        rec2.at(kPY + slot) = zp.y;
        rec2.at(kW + slot) = w;
      }
    }
  }
  if (nreal == 3) {   // ghost pair positions for the slope detector
    rec.at(kZX + 1) = eA.x + L.z2;
    rec.at(kZY + 1) = eA.y;
    rec.at(kZX + 4) = eB.x + L.z2;
    rec.at(kZY + 4) = eB.y;
    if (kDual) {
      rec2.at(kZX + 1) = eA.x + L.z2;
      rec2.at(kZY + 1) = eA.y;
      rec2.at(kZX + 4) = eB.x + L.z2;
      rec2.at(kZY + 4) = eB.y;
    }
  }
  rec.set_code(nreal + 8 * flags);
  if (kDual) rec2.set_code(nreal + 8 * flags);
  if (out_count) *out_count = (int8_t)nreal;
  return flags;
}

// Seed block of one source (kSeedDoubles doubles, element e at seeds[e * stride]):
//   [0..4] Re eta_k, [5..9] Im eta_k   the five planet-frame roots of the point source at the source CENTRE (cold solve)
//   [10..14] Re(A_k + B_k), [15..19] Im(B_k - A_k), [20..24] Im(A_k + B_k), [25..29] Re(A_k - B_k)
//                                      first-order response of root k to a displacement delta of the source,
//                                      d eta_k = A_k delta + B_k conj(delta), stored as the real 2 x 2 map of
//                                      (Re delta, Im delta) -> (Re d eta_k, Im d eta_k): four FMAs per root and sample
//   [30]                               1 when two roots are closer than 1e-6 of the roots' scale (next to a planet of
//                                      tiny q): the seeded solve then also verifies the PRODUCT of the roots
// The quintic's roots are the fixed points (real images) and the 2-cycle (ghost pair) of T(z) = zeta - conj f(z)
// (G-1): z_a = zeta - conj f(z_b), z_b = zeta - conj f(z_a), with z_b = z_a for a real image.
// Differentiating both and eliminating dz_b gives dz_a (1 - f'(w_a) f'(z_a)) = delta - f'(w_a) conj(delta) with
// w_a = conj(z_b) = conj(zeta) - f(z_a); conj(f'(z_b)) = f'(conj z_b) because both lenses are on the real axis.  For
// a real image this is Eq.(10)'s z'.  A prediction is kept only when the shift rho (|A| + |B|) stays below
// a quarter of the distance to the nearest other root (next to a caustic 1/J blows up); otherwise A = B = 0.
constexpr int kSeedDoubles = 31;

// Element e goes to seeds[e * stride] (stride > 0) or, for the [kSeedDoubles][n] workspace layout, to seeds[e * wide]
// (stride == 0).
TWK_HD void centre_seeds(const Lens& L, cd zc, double rho, double* seeds, int stride, long long wide = 0) {
  const size_t st = stride > 0 ? (size_t)stride : (size_t)wide;
  cd c[6], eta[5];
  double dmin2_all = 1e300;
  cd y = mk(zc.x - L.z2, zc.y);
  lens_guard(y, L.s);   // a source CENTRE on a lens is an ordinary input (the disk covers the lens)
  coeffs_eq6(y, L.s, L.m2, c);
  {
    Coef6 C;
#pragma unroll
    for (int i = 0; i < 6; ++i) C.c[i] = c[i];
    const Roots5 R = quintic_roots_cold(C);
#pragma unroll
    for (int k = 0; k < 5; ++k) eta[k] = R.r[k];
  }
  {   // the root of largest modulus goes last: the seeded solve derives the fifth root from Vieta's sum (twk_device.cuh)
    int big = 0;
    double nb = norm2(eta[0]);
#pragma unroll
    for (int k = 1; k < 5; ++k)
      if (norm2(eta[k]) > nb) { nb = norm2(eta[k]); big = k; }
    const cd last = eta[4];
    cd e = eta[0];
#pragma unroll
    for (int k = 1; k < 5; ++k)
      if (k == big) e = eta[k];
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (k == big) eta[k] = last;
    eta[4] = e;
  }
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const cd a = crecip(mk(-L.s - eta[k].x, -eta[k].y));
    const cd b = crecip(-eta[k]);
    const cd f = L.m1 * a + L.m2 * b;
    const cd fz = L.m1 * (a * a) + L.m2 * (b * b);
    const cd w = mk(y.x - f.x, -y.y - f.y);                    // conj(eta_b) = conj(y) - f(z_a), planet frame
    const cd aw = crecip(mk(-L.s - w.x, -w.y));
    const cd bw = crecip(-w);
    const cd fw = L.m1 * (aw * aw) + L.m2 * (bw * bw);
    const cd den = mk(1.0, 0.0) - fw * fz;
    cd A = crecip(den);
    cd B = -(fw * A);
    double dmin2 = 1e300;
#pragma unroll
    for (int j = 0; j < 5; ++j)
      if (j != k) dmin2 = fmin(dmin2, norm2(eta[k] - eta[j]));
    const double shift = rho * (sqrt(norm2(A)) + sqrt(norm2(B)));
    if (!(shift * shift <= 0.0625 * dmin2)) {                   // also catches NaN / inf
      A = mk(0.0, 0.0);
      B = mk(0.0, 0.0);
    }
    dmin2_all = fmin(dmin2_all, dmin2);
    seeds[k * st] = eta[k].x;
    seeds[(5 + k) * st] = eta[k].y;
    // A delta + B conj(delta) = (A.x + B.x) dx + (B.y - A.y) dy + i [(A.y + B.y) dx + (A.x - B.x) dy]
    seeds[(10 + k) * st] = A.x + B.x;
    seeds[(15 + k) * st] = B.y - A.y;
    seeds[(20 + k) * st] = A.y + B.y;
    seeds[(25 + k) * st] = A.x - B.x;
  }
  const double scale = abs1(eta[0]) + abs1(eta[1]) + abs1(eta[2]) + abs1(eta[3]) + abs1(eta[4]);
  seeds[30 * st] = (dmin2_all < 1e-12 * scale * scale) ? 1.0 : 0.0;
}

// ------------------------------------------------------------------------------------------------------------
// N1: point-source adequacy tests in front of the contour path ("the quadrupole test and ghost
// image test check if the point-source approximation is accurate enough").  The paper gives no formulas; these are
// derived here (readings N1-a..c) from the lens equation alone:
//  * a uniform disk of radius rho sees  mu_fs = mu + (rho^2 / 8) Laplacian(mu) + O(rho^4),  Laplacian = 4 d^2/dzeta dzetabar;
//    for one image with g = f1(z), h = f2(z), k = f3(z) (first, second, third derivative of f), J = 1 - g gbar, the
//    chain rule through dz/dzeta = 1/J, dz/dzetabar = -gbar/J gives  d(1/J)/dzeta = N / J^3,  N = h gbar - g^2 hbar,
//    and  d^2(1/J)/dzeta dzetabar = [ -gbar (N_z/J^3 - 3 N J_z/J^4) + (N_zb/J^3 - 3 N J_zb/J^4) ] / J  with
//    N_z = k gbar - 2 g h hbar, N_zb = h hbar - g^2 kbar, J_z = -h gbar, J_zb = -g hbar;
//    the same operator once more in zeta gives the traceless second derivative d^2(1/J)/dzeta^2 = (M_z - g M_zb)/J,
//    M = N/J^3.  The disk average keeps only the Laplacian, but next to a cusp the Laplacian of a bright image
//    changes sign while the traceless part stays large, so the test bounds both;
//  * quadrupole test: sum over real images of rho^2/2 (|d2/dzeta dzetabar| + |d2/dzeta^2|) of 1/J < kPsQuad * tol * A;
//  * ghost-image test: a ghost root moves by A_k delta + B_k conj(delta) (centre_seeds); the pair merges into a real
//    pair when the two close their separation |R_k| (the 2-cycle step): require rho (|A_k| + |B_k|) < kPsGhost |R_k|.
// Returns true when both tests pass; mu = A + quadrupole term, qrel = the size of the quadrupole term relative to A.
// ------------------------------------------------------------------------------------------------------------
constexpr double kPsQuad = 3.0;    // reading N1-b: calibrated against the converged contour values of the oracle
constexpr double kPsGhost = 0.1;   // reading N1-c

TWK_HD bool point_source_adequate(const Lens& L, cd zc, double rho, const double* seeds, int stride, double tol, double& mu,
                                  double& qrel) {
  cd y = mk(zc.x - L.z2, zc.y);
  lens_guard(y, L.s);
  cd eta[5], g[5], f[5], Res[5];
  double R2[5];
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    eta[k] = mk(seeds[k * stride], seeds[(5 + k) * stride]);
    const cd a = crecip(mk(-L.s - eta[k].x, -eta[k].y));
    const cd b = crecip(-eta[k]);
    f[k] = L.m1 * a + L.m2 * b;
    g[k] = L.m1 * (a * a) + L.m2 * (b * b);
    Res[k] = mk(y.x - eta[k].x - f[k].x, y.y - eta[k].y + f[k].y);
    R2[k] = norm2(Res[k]);
  }
  // residual detector, as in point_solve_cs
  // (running maxima in scalars: no dynamically indexed array, everything stays in registers)
  int ia = 0, ib = -1;
  double mA = R2[0], mB = -1.0;
  cd eA = eta[0], rA = Res[0], eB = eta[0], rB = Res[0];
#pragma unroll
  for (int k = 1; k < 5; ++k) {
    if (R2[k] > mA) {          // new largest: the old largest becomes the second
      mB = mA; ib = ia; eB = eA; rB = rA;
      mA = R2[k]; ia = k; eA = eta[k]; rA = Res[k];
    } else if (R2[k] > mB) {
      mB = R2[k]; ib = k; eB = eta[k]; rB = Res[k];
    }
  }
  const cd dab = eB - eA;
  const bool ghost = norm2(rA - dab) < mA && norm2(rB + dab) < mB;
  double A = 0.0, Q = 0.0, Qabs = 0.0;
  int npos = 0, nreal = 0;
  bool ok = true;
  const double hr2 = 0.5 * rho * rho;
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const cd a = crecip(mk(-L.s - eta[k].x, -eta[k].y));
    const cd b = crecip(-eta[k]);
    const cd a2 = a * a, b2 = b * b;
    if (ghost && (k == ia || k == ib)) {
      // ghost-image test: response of the ghost root, A = 1/D, B = -f1(w)/D, D = 1 - f1(w) f1(z), w = conj(y) - f(z)
      const cd w = mk(y.x - f[k].x, -y.y - f[k].y);
      const cd aw = crecip(mk(-L.s - w.x, -w.y));
      const cd bw = crecip(-w);
      const cd gw = L.m1 * (aw * aw) + L.m2 * (bw * bw);
      const cd D = mk(1.0, 0.0) - gw * g[k];
      const double resp = (1.0 + sqrt(norm2(gw))) * sqrt(rcp(norm2(D)));   // |A| + |B|
      ok = ok && (rho * resp < kPsGhost * sqrt(R2[k]));
      continue;
    }
    const cd h = 2.0 * (L.m1 * (a2 * a) + L.m2 * (b2 * b));
    const cd kk = 6.0 * (L.m1 * (a2 * a2) + L.m2 * (b2 * b2));
    const cd gb = conj(g[k]), hb = conj(h), kb = conj(kk);
    const double J = 1.0 - norm2(g[k]);
    const double iJ = rcp(J), iJ3 = iJ * iJ * iJ, iJ4 = iJ3 * iJ;
    const cd g2 = g[k] * g[k];
    const cd N = h * gb - g2 * hb;
    const cd Nz = kk * gb - 2.0 * ((g[k] * h) * hb);
    const cd Nzb = h * hb - g2 * kb;
    const cd Jz = -(h * gb), Jzb = -(g[k] * hb);
    const cd Mz = iJ3 * Nz - (3.0 * iJ4) * (N * Jz);
    const cd Mzb = iJ3 * Nzb - (3.0 * iJ4) * (N * Jzb);
    const cd mzz = iJ * (Mzb - gb * Mz);                  // d2(1/J) / dzeta dzetabar  (a quarter of the Laplacian)
    const cd mz2 = iJ * (Mz - g[k] * Mzb);                // d2(1/J) / dzeta^2         (the traceless part)
    const double p = (J > 0.0) ? 1.0 : -1.0;
    A += p * iJ;
    Q += p * hr2 * mzz.x;
    Qabs += hr2 * (sqrt(norm2(mzz)) + sqrt(norm2(mz2)));
    npos += (J > 0.0);
    ++nreal;
  }
  ok = ok && (npos == ((nreal - 1) >> 1));             // parity sum -1; no repair here: leave it to the contour
  mu = A + Q;
  qrel = Qabs * rcp(fabs(A));
  return ok && isfinite(mu) && isfinite(qrel) && (Qabs < kPsQuad * tol * fabs(A));
}

// out-of-line entry (once per source, outside the hot loop: keeps its registers and code away from it)
struct PsResult {
  double mu, qrel;
  int ok;
};
TWK_NOINLINE PsResult point_source_adequate_cold(Lens L, cd zc, double rho, const double* seeds, int stride, double tol) {
  PsResult r;
  r.ok = point_source_adequate(L, zc, rho, seeds, stride, tol, r.mu, r.qrel) ? 1 : 0;
  return r;
}

// ------------------------------------------------------------------------------------------------------------
// a6 + a7: one interval theta_A -> theta_B (dth = theta_B - theta_A > 0).
// ------------------------------------------------------------------------------------------------------------
struct Piece {
  double dA, err;
  int crossing;   // 0 none, +1 creation, -1 annihilation
  int slope;      // slope detector (a5): 0 fine; otherwise the crossing's real pair is NOT perpendicular to the
                  // ghost pair next to it and must be re-judged: slot of its positive image | slot of its negative << 4 | 256
};

// the powers of the interval's width that every link of the interval uses (computed once per interval)
struct LinkConst {
  double dth2, c24, c12, c48;   // dth^2, dth^3/24, dth/12, dth^3/48
};
TWK_HD LinkConst link_const(double dth) {
  LinkConst K;
  K.dth2 = dth * dth;
  const double dth3 = K.dth2 * dth;
  K.c24 = dth3 * (1.0 / 24.0);
  K.c12 = dth * (1.0 / 12.0);
  K.c48 = dth3 * (1.0 / 48.0);
  return K;
}
TWK_HD void link_terms(const RecRef& A, const RecRef& B, int ka, int kb, double par, const LinkConst& K, double& dA,
                       double& err) {
  const cd zA = A.z(ka), zB = B.z(kb), pA = A.zp(ka), pB = B.zp(kb);
  const double wA = A.w(ka), wB = B.w(kb);
  const cd dz = zB - zA;
  const double trap = 0.5 * wedge(zA, dz);                              // Eq.(9)
  const double p1 = (wA + wB) * K.c24;                                  // Eq.(10) dA^(p1)
  const double p2 = wedge(dz, pB - pA) * K.c12;                         // Eq.(10) dA^(p2)
  const double dAp = 0.5 * (p1 + p2);
  dA += par * (trap + dAp);
  const double E1 = fabs(wA - wB) * K.c48;                              // Eq.(17)
  const double E2 = 1.5 * fabs(dAp * (norm2(dz) * rcp1(K.dth2 * fabs(dotp(pA, pB))) - 1.0));   // (an estimate: 40 bits do)
  const double E3 = 0.1 * fabs(dAp) * K.dth2;
  const double E4 = fabs(p1 - p2);
  err += (E1 + E2) + (E3 + E4);
}

// 2 x 2 minimum-total-distance matching from SQUARED distances: returns 1 when the crossed pairing (0-1, 1-0) is
// shorter than the straight one (0-0, 1-1); ties keep the straight pairing (reading L-3).  Short cut without square
// roots: 2 (s00 + s11) < min(s01, s10) gives sqrt s00 + sqrt s11 <= sqrt(2 (s00 + s11)) < sqrt(min) <= sqrt s01 + sqrt s10,
// so the straight pairing is the shorter one (and the mirror statement); the decision is the exact one whenever the
// short cut applies, and it applies unless the images are about as close to each other as to their successors.
TWK_HD int crossed_is_shorter(double s00, double s11, double s01, double s10) {
  const double st = 2.0 * (s00 + s11), cr = 2.0 * (s01 + s10);
  if (st < s01 && st < s10) return 0;
  if (cr < s00 && cr < s11) return 1;
  return (sqrt(s01) + sqrt(s10)) < (sqrt(s00) + sqrt(s11));
}

// K = link_const(dth) of the interval's width dth = theta_B - theta_A > 0
TWK_HD Piece eval_interval(const RecRef& A, const RecRef& B, const LinkConst& K, double slope_gate2, double slope_cos2) {
  Piece P;
  P.dA = 0.0;
  P.err = 0.0;
  P.crossing = 0;
  P.slope = 0;
  const bool a5 = A.nreal() == 5, b5 = B.nreal() == 5;
  int leftApos = -1, leftAneg = -1, leftBpos = -1, leftBneg = -1;
  // links are collected first (slot of A | slot of B << 3, six bits each: five links fit one 32-bit word) and evaluated
  // in ONE loop below
  unsigned links = 0;
  int nl = 0;
  auto add_link = [&](int ka, int kb) {
    links |= (unsigned)(ka | (kb << 3)) << (6 * nl);
    ++nl;
  };
  // ---- positive parity: slots 0,(1) --------------------------------------------------------------------
  {
    const cd A0 = A.z(0), B0 = B.z(0);
    if (!a5 && !b5) {
      add_link(0, 0);
    } else if (a5 && b5) {
      const cd A1 = A.z(1), B1 = B.z(1);
      const int sw = crossed_is_shorter(norm2(A0 - B0), norm2(A1 - B1), norm2(A0 - B1), norm2(A1 - B0));
      add_link(0, sw);
      add_link(1, 1 - sw);
    } else if (b5) {   // 1 -> 2: the nearer one links, the other is left over
      const int j = norm2(A0 - B.z(1)) < norm2(A0 - B0);
      add_link(0, j);
      leftBpos = 1 - j;
    } else {           // 2 -> 1
      const int i = norm2(A.z(1) - B0) < norm2(A0 - B0);
      add_link(i, 0);
      leftApos = 1 - i;
    }
  }
  // ---- negative parity: slots 2,3,(4): minimum-total-distance injective matching -----------------
  if (!a5 && !b5) {
    const cd A2 = A.z(2), A3 = A.z(3), B2 = B.z(2), B3 = B.z(3);
    const int sw = crossed_is_shorter(norm2(A2 - B2), norm2(A3 - B3), norm2(A2 - B3), norm2(A3 - B2));
    add_link(2, 2 + sw);
    add_link(3, 3 - sw);
  } else {
    const int na = a5 ? 3 : 2, nb = b5 ? 3 : 2;
    double D[3][3];
    cd za[3], zb[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      za[i] = (i < na) ? A.z(2 + i) : mk(0.0, 0.0);
      zb[i] = (i < nb) ? B.z(2 + i) : mk(0.0, 0.0);
    }
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const bool ra = i < na, rb = j < nb;
        // a missing third image is a dummy: free against real images (only one side lacks it here)
        D[i][j] = (ra && rb) ? sqrt(norm2(za[i] - zb[j])) : 0.0;
      }
    const int perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    int bestp = 0;
    double best = D[0][0] + D[1][1] + D[2][2];
#pragma unroll
    for (int p = 1; p < 6; ++p) {
      const double cost = D[0][perm[p][0]] + D[1][perm[p][1]] + D[2][perm[p][2]];
      if (cost < best) { best = cost; bestp = p; }
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      int j = 0;
#pragma unroll
      for (int p = 0; p < 6; ++p)
        if (p == bestp) j = perm[p][i];
      const bool ra = i < na, rb = j < nb;
      if (ra && rb) add_link(2 + i, 2 + j);
      else if (ra) leftAneg = 2 + i;
      else if (rb) leftBneg = 2 + j;
    }
  }
  // ---- a7: area and error of every link (one copy of the code; 3 or 4 or 5 trips) ----------------------------
#pragma unroll 1
  for (int l = 0; l < nl; ++l) {
    const int ka = (int)(links & 7u), kb = (int)((links >> 3) & 7u);
    links >>= 6;
    link_terms(A, B, ka, kb, ka < 2 ? 1.0 : -1.0, K, P.dA, P.err);
  }
  // ---- caustic crossing: the extra (+,-) pair on the 5-image side connects to itself -------------
  if (a5 != b5) {
    const bool creation = b5;
    const RecRef& S = creation ? B : A;
    const int kp = creation ? leftBpos : leftApos;
    const int km = creation ? leftBneg : leftAneg;
    const cd zpl = S.z(kp), zmi = S.z(km), ppl = S.zp(kp), pmi = S.zp(km);
    const double wpl = S.w(kp), wmi = S.w(km);
    const cd d = zpl - zmi;
    {
      // a5, slope detector (reading G-4): next to the critical curve the real pair of the 5-image sample
      // and the ghost pair of the 3-image sample point in perpendicular directions.  Applied only when both pairs
      // are closer than the gate (the local expansion of Eq.(16) holds near the critical curve only
      // "works only for the point sources near caustics"); not perpendicular (|cos| >= slope_cos, 45 deg by
      // default) = misjudged.
      const RecRef& G = creation ? A : B;
      const cd dg = G.z(1) - G.z(4);
      const double n_r = norm2(d), n_g = norm2(dg), c = dotp(d, dg);
      if (n_r < slope_gate2 && n_g < slope_gate2 && c * c >= slope_cos2 * n_r * n_g) P.slope = kp | (km << 4) | 256;
    }
    const double ad = sqrt(norm2(d));
    const double sq = sqrt(fabs(dotp(ppl, pmi)));
    const double dtt = ad / sq;                                         // Eq.(11) tilde Delta theta
    const double dtt3 = dtt * dtt * dtt;
    const double corr = (wpl - wmi) * dtt3 * (1.0 / 24.0);              // Eq.(11)
    const double dd = dotp(d, ppl - pmi);
    // Eq.(11) enters as printed in both directions (S-2): the pair's path runs z- -> z+ at a creation and
    // z+ -> z- at an annihilation; only the closing chord and the sign rule of E2 depend on the direction
    const double dAp = corr;
    const double chord = creation ? 0.5 * wedge(zmi, d) : -0.5 * wedge(zpl, d);
    const double E2 = 1.5 * fabs(creation ? dd - 2.0 * ad * sq : dd + 2.0 * ad * sq) * dtt;   // Eq.(18), reading E-5
    P.crossing = creation ? 1 : -1;
    P.dA += chord + dAp;
    const double E1 = fabs(wpl + wmi) * dtt3 * (1.0 / 48.0);            // Eq.(18)
    const double E3 = 0.1 * fabs(dAp) * K.dth2;
    P.err += E1 + E2 + E3;
  }
  return P;
}
TWK_HD Piece eval_interval(const RecRef& A, const RecRef& B, double dth, double slope_gate2, double slope_cos2) {
  return eval_interval(A, B, link_const(dth), slope_gate2, slope_cos2);
}

// ------------------------------------------------------------------------------------------------------------
// L-4 guard (an EXTENSION of the paper's estimate, option hidden_crossing_guard, off by default; reading L-4).
// Eq.(17) sees an interval through its end points only: a boundary that dips into a caustic and out again BETWEEN two
// adjacent 3-image samples leaves no trace in them.  The ghost pair does: next to a fold its separation squared
// D = |z_a - z_b|^2 is proportional to the distance of the boundary point from the caustic, a parabola in theta that
// turns negative where the boundary is inside.  D is fitted through (A-, A, B) and (A, B, B+); a convex fit with its
// vertex inside the interval at D* < 0 is a hidden pair of crossings enclosing the area v (pi/2)(-D*)/sqrt(C) (C = the
// fit's curvature, v = speed of the ghost pair's midpoint); that area is added to the interval's error estimate.
// dm, d, dp = theta_A - theta_A-, theta_B - theta_A, theta_B+ - theta_B.  Out of line: rare, optional.
// ------------------------------------------------------------------------------------------------------------
TWK_NOINLINE double hidden_crossing_term(RecRef Am, RecRef A, RecRef B, RecRef Bp, double dm, double d, double dp) {
  if (A.nreal() != 3 || B.nreal() != 3) return 0.0;
  const cd sA = A.z(1) - A.z(4), sB = B.z(1) - B.z(4);
  const cd mA = A.z(1) + A.z(4), mB = B.z(1) + B.z(4);            // twice the midpoints
  const double DA = norm2(sA), DB = norm2(sB);
  const double v = 0.5 * sqrt(norm2(mB - mA)) / d;
  double term = 0.0;
#pragma unroll 1
  for (int side = 0; side < 2; ++side) {
    const RecRef& T = side ? Bp : Am;
    if (T.nreal() != 3) continue;
    const double D3 = norm2(T.z(1) - T.z(4));
    const double x0 = side ? 0.0 : -dm, x1 = side ? d : 0.0, x2 = side ? d + dp : d;
    const double y0 = side ? DA : D3, y1 = side ? DB : DA, y2 = side ? D3 : DB;
    const double f01 = (y1 - y0) / (x1 - x0), f12 = (y2 - y1) / (x2 - x1);
    const double C = (f12 - f01) / (x2 - x0);
    if (!(C > 0.0)) continue;
    const double xs = 0.5 * (x0 + x1) - f01 / (2.0 * C);
    if (!(xs > 0.0 && xs < d)) continue;
    const double ys = y0 + f01 * (xs - x0) + C * (xs - x0) * (xs - x1);
    if (!(ys < 0.0)) continue;
    term = fmax(term, v * (0.5 * 3.141592653589793238462643383279) * (-ys) / sqrt(C));
  }
  return term;
}

// a5, slope detector: re-judge the real pair (slots kp, km) of a 5-image record as the ghost pair ("pair 1
// shall be rejudged as ghost images").  The record becomes a 3-image record: the other positive image in slot 0, the
// other two negative images in slots 2 and 3, the pair's positions in the z fields of slots 1 and 4.
TWK_HD void demote_pair(const RecRef& S, int kp, int km) {
  const cd gp = S.z(kp), gm = S.z(km);
  if (kp == 0) {
    S.at(kZX) = S.at(kZX + 1);
    S.at(kZY) = S.at(kZY + 1);
    S.at(kPX) = S.at(kPX + 1);
    S.at(kPY) = S.at(kPY + 1);
    S.at(kW) = S.at(kW + 1);
  }
  if (km < 4) {   // slot 4 moves down into the hole
    S.at(kZX + km) = S.at(kZX + 4);
    S.at(kZY + km) = S.at(kZY + 4);
    S.at(kPX + km) = S.at(kPX + 4);
    S.at(kPY + km) = S.at(kPY + 4);
    S.at(kW + km) = S.at(kW + 4);
  }
  S.at(kZX + 1) = gp.x;
  S.at(kZY + 1) = gp.y;
  S.at(kZX + 4) = gm.x;
  S.at(kZY + 4) = gm.y;
  S.set_code(3 + 8 * (S.point_flags() | kPointSlope));
}

}  // namespace twk
