// twk_device.cuh -- device functions of the hot path, rows a1-a7 of SURVEY.md section 8(a).
//
//   a1  boundary sample            zeta_j = zeta_c + rho e^{i theta_j}, zeta'_j = i rho e^{i theta_j}
//   a2  coefficient builder        Eq.(6), planet frame
//   a3  quintic solve              seeded Newton on the full polynomial (Vieta-verified, Vieta recovery); cold solver:
//                                  Laguerre + forward deflation + Newton polish
//   a4  per-root lens quantities   f', f'', R (Eq.12), J (Eq.7), z' and z'^z'' (Eq.10, repaired)
//   a5  ghost filter               residual detector, 2-cycle reading; slope detector at count changes
//   a6  contour linker             per-parity minimum-total-distance matching, creation / annihilation
//   a7  area + error per interval  Eq.(9)-(11), Eq.(17)-(18)
//
// "P:<n>" = /root/reference/PAPER.md line n.  Nothing here is shared with oracle/ (which uses a different
// root finder and enumerates permutations with the standard library).
//
// TWK_HD is __device__ in the product build.  (A host build of these functions exists only in throw-away
// probes, never in the library.)
#pragma once

#include <math.h>
#include <stdint.h>

#ifndef TWK_HD
#define TWK_HD __device__ __forceinline__
#endif
#ifndef TWK_NOINLINE
#define TWK_NOINLINE __device__ __noinline__   // rarely executed paths stay out of the hot instruction stream
#endif
#ifndef TWK_COUNT
#define TWK_COUNT(what)   // event counter hook of the host-side probes; nothing in the library
#endif

namespace twk {

// ------------------------------------------------------------------------------------------------------------
// complex FP64 arithmetic on register pairs
// ------------------------------------------------------------------------------------------------------------
struct cd {
  double x, y;
};
TWK_HD cd mk(double x, double y) { cd r; r.x = x; r.y = y; return r; }
TWK_HD cd operator+(cd a, cd b) { return mk(a.x + b.x, a.y + b.y); }
TWK_HD cd operator-(cd a, cd b) { return mk(a.x - b.x, a.y - b.y); }
TWK_HD cd operator-(cd a) { return mk(-a.x, -a.y); }
TWK_HD cd operator*(cd a, cd b) { return mk(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x)); }
TWK_HD cd operator*(double s, cd a) { return mk(s * a.x, s * a.y); }
TWK_HD cd conj(cd a) { return mk(a.x, -a.y); }
TWK_HD double norm2(cd a) { return fma(a.x, a.x, a.y * a.y); }
TWK_HD double abs1(cd a) { return fabs(a.x) + fabs(a.y); }
TWK_HD double wedge(cd a, cd b) { return fma(a.x, b.y, -(a.y * b.x)); }
TWK_HD double dotp(cd a, cd b) { return fma(a.x, b.x, a.y * b.y); }
TWK_HD cd cfma(cd a, cd b, cd c) {                                        // a*b + c
  return mk(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y)));
}
// 1/x for a normal, finite x: the hardware's 20-bit estimate + two Newton steps (5 instructions, ~1 ulp) instead of
// the IEEE-rounded division with its range checks (~12).  x = 0 or non-finite gives inf or NaN, which every caller
// tolerates (guards on the denominator or the kPointNonFinite flag).
TWK_HD double rcp(double x) {
#ifdef __CUDA_ARCH__
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, e, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
#else
  return 1.0 / x;
#endif
}
// 1/x to ~40 bits: the estimate + ONE Newton step.  For Newton corrections only (a relative error of 1e-12 in a step
// that is itself <= 1e-4 of the root is far below the rounding of the root).
TWK_HD double rcp1(double x) {
#ifdef __CUDA_ARCH__
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);
  return fma(y, e, y);
#else
  return 1.0 / x;
#endif
}
TWK_HD cd crecip(cd a) {
  const double inv = rcp(norm2(a));
  return mk(a.x * inv, -a.y * inv);
}
TWK_HD cd cdiv(cd a, cd b) {
  const double inv = rcp(norm2(b));
  return mk(fma(a.x, b.x, a.y * b.y) * inv, fma(a.y, b.x, -(a.x * b.y)) * inv);
}
TWK_HD cd csqrt_(cd a) {   // principal square root
  const double r = sqrt(norm2(a));
  if (r == 0.0) return mk(0.0, 0.0);
  const double t = sqrt(0.5 * (r + fabs(a.x)));
  const double u = 0.5 * a.y / t;
  return (a.x >= 0.0) ? mk(t, u) : mk(fabs(u), copysign(t, a.y));
}

// ------------------------------------------------------------------------------------------------------------
// lens geometry, Eq.(2)
// ------------------------------------------------------------------------------------------------------------
struct Lens {
  double s, m1, m2, z2;   // separation, masses normalised to the total, secondary position (CM frame)
};
TWK_HD Lens make_lens(double s, double q) {
  Lens L;
  const double inv = 1.0 / (1.0 + q);
  L.s = s;
  L.m1 = inv;
  L.m2 = q * inv;
  L.z2 = s * inv;
  return L;
}

// ------------------------------------------------------------------------------------------------------------
// a2. Eq.(6): cancellation-free coefficients in the planet frame (planet at 0, primary at -s).
//     y = zeta - z2, v_c = conj(y) + s, v_p = 1 + s conj(y).
// ------------------------------------------------------------------------------------------------------------
TWK_HD void coeffs_eq6(cd y, double s, double m2, cd c[6]) {
  const cd yb = conj(y);
  const cd vc = mk(yb.x + s, yb.y);
  const cd vp = mk(fma(s, yb.x, 1.0), s * yb.y);
  const double Iy = y.y;
  const double m2s = m2 * s;
  const double yy = norm2(y);   // conj(y) y
  // c5 = -conj(y) v_c
  c[5] = -(yb * vc);
  // c4 = (conj(y) y - 1 - 2 s conj(y)) v_c + m2 s
  {
    const cd t = mk(yy - 1.0 - 2.0 * s * yb.x, -2.0 * s * yb.y);
    c[4] = cfma(t, vc, mk(m2s, 0.0));
  }
  // c3 = (2y - s) [v_p v_c + 2 i Im y - m2 s] + 4 i (m2 s - y) Im y
  {
    const cd a = mk(2.0 * y.x - s, 2.0 * y.y);
    const cd b = cfma(vp, vc, mk(-m2s, 2.0 * Iy));
    const cd d = mk(m2s - y.x, -y.y);           // (m2 s - y)
    const cd e = mk(-4.0 * Iy * d.y, 4.0 * Iy * d.x);   // 4 i Im(y) (m2 s - y)
    c[3] = cfma(a, b, e);
  }
  // c2 = Re(v_p)^2 Re(v_c) + i Im(y) Re(v_p) Re(1 - s y) + s Im(y)^2 (2 + s v_c) + m2 s [2 conj(y)(y - s) - (1 - s y)]
  {
    const double rvp = vp.x, rvc = vc.x;
    const cd t3 = mk(2.0 + s * vc.x, s * vc.y);
    const cd ys = mk(y.x - s, y.y);
    const cd br = 2.0 * (yb * ys) - mk(1.0 - s * y.x, -s * y.y);
    c[2] = mk(rvp * rvp * rvc + s * Iy * Iy * t3.x + m2s * br.x,
              Iy * rvp * (1.0 - s * y.x) + s * Iy * Iy * t3.y + m2s * br.y);
  }
  // c1 = m2 s [(s + 2y) v_p + s (2 i s Im y - m2)]
  {
    const cd a = mk(s + 2.0 * y.x, 2.0 * y.y);
    const cd t = cfma(a, vp, mk(-s * m2, 2.0 * s * s * Iy));
    c[1] = m2s * t;
  }
  // c0 = s^2 m2^2 y
  c[0] = (m2s * m2s) * y;
}

// ------------------------------------------------------------------------------------------------------------
// a3. quintic roots.  Laguerre iteration from x = 0 on the successively (forward-)deflated polynomial for the
// first three roots, closed form for the remaining quadratic, then Newton steps on the ORIGINAL polynomial for
// all five (removes deflation error).  All in registers; loops are compile-time bounded.
// ------------------------------------------------------------------------------------------------------------
constexpr double kEps = 2.220446049250313e-16;
#ifndef TWK_STOP_FACTOR
#define TWK_STOP_FACTOR 450.0   // Newton stop rule: predicted next step <= TWK_STOP_FACTOR * eps * |root| = 1e-13 |root|
#endif

template <int N>
TWK_HD cd laguerre(const cd (&a)[N + 1], cd x) {
  double a1[N + 1];
#pragma unroll
  for (int i = 0; i <= N; ++i) a1[i] = abs1(a[i]);
  double last = 1e300;
  for (int it = 0; it < 48; ++it) {
    cd p = a[N], d = mk(0.0, 0.0), h = mk(0.0, 0.0);   // p, p', p''/2
    double err = a1[N];
    const double ax = abs1(x);
#pragma unroll
    for (int i = N - 1; i >= 0; --i) {
      h = cfma(h, x, d);
      d = cfma(d, x, p);
      p = cfma(p, x, a[i]);
      err = fma(err, ax, a1[i]);
    }
    if (abs1(p) <= 2.0 * kEps * err) break;           // at the rounding floor of the evaluation
    // dx = N p / (p' +- sqrt((N-1)((N-1) p'^2 - 2 N p p''/2)))
    const cd g2 = d * d;
    const cd ph = p * h;
    const cd rad = mk(double(N - 1) * (double(N - 1) * g2.x - double(2 * N) * ph.x),
                      double(N - 1) * (double(N - 1) * g2.y - double(2 * N) * ph.y));
    cd sq = csqrt_(rad);
    if (dotp(d, sq) < 0.0) sq = -sq;
    const cd den = d + sq;
    cd dx;
    if (norm2(den) > 0.0) dx = cdiv(double(N) * p, den);
    else dx = mk((1.0 + ax) * cos(double(it + 1)), (1.0 + ax) * sin(double(it + 1)));
    const double sdx = abs1(dx);
    if ((it & 7) == 7 && sdx >= last) dx = 0.5 * dx;   // break rare limit cycles
    last = sdx;
    x = x - dx;
    if (sdx <= kEps * abs1(x)) break;
  }
  return x;
}

template <int N>
TWK_HD void deflate(const cd (&a)[N + 1], cd r, cd (&b)[N]) {
  b[N - 1] = a[N];
#pragma unroll
  for (int i = N - 1; i >= 1; --i) b[i - 1] = cfma(r, b[i], a[i]);
}

TWK_HD void quadratic(const cd (&a)[3], cd& r0, cd& r1) {
  const cd disc = a[1] * a[1] - 4.0 * (a[2] * a[0]);
  cd sq = csqrt_(disc);
  if (dotp(a[1], sq) < 0.0) sq = -sq;
  const cd qq = -0.5 * (a[1] + sq);
  if (norm2(qq) > 0.0) {
    r0 = cdiv(qq, a[2]);
    r1 = cdiv(a[0], qq);
  } else {
    r0 = mk(0.0, 0.0);
    r1 = mk(0.0, 0.0);
  }
}

TWK_HD void quintic_roots(const cd (&c)[6], cd (&r)[5]) {
  cd b4[5], b3[4], b2[3];
  r[0] = laguerre<5>(c, mk(0.0, 0.0));
  deflate<5>(c, r[0], b4);
  r[1] = laguerre<4>(b4, mk(0.0, 0.0));
  deflate<4>(b4, r[1], b3);
  r[2] = laguerre<3>(b3, mk(0.0, 0.0));
  deflate<3>(b3, r[2], b2);
  quadratic(b2, r[3], r[4]);
  // Newton polish on the undeflated quintic: two steps per root, five independent chains (ILP)
#pragma unroll
  for (int pass = 0; pass < 2; ++pass) {
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      cd p = c[5], d = mk(0.0, 0.0);
#pragma unroll
      for (int i = 4; i >= 0; --i) {
        d = cfma(d, r[k], p);
        p = cfma(p, r[k], c[i]);
      }
      const double dn = norm2(d);
      if (dn > 0.0) {
        const cd dx = cdiv(p, d);
        // never let a polish step move a root by more than its own size (guards a vanishing p')
        if (norm2(dx) <= norm2(r[k]) + 1e-300) r[k] = r[k] - dx;
      }
    }
  }
}

// The cold solver as an out-of-line call (arguments and result by value, so the caller's coefficient and root
// registers never have their address taken): it is the rare fallback of the seeded solve, and ~6 k instructions
// that must not sit in the middle of the hot loop's instruction stream.
struct Coef6 { cd c[6]; };
struct Roots5 { cd r[5]; };
TWK_NOINLINE Coef6 coeffs_eq6_cold(cd y, double s, double m2) {   // (rebuilt after the B-1 guard moved y: rare)
  Coef6 C;
  coeffs_eq6(y, s, m2, C.c);
  return C;
}
TWK_NOINLINE Roots5 quintic_roots_cold(Coef6 C) {
  Roots5 R;
  quintic_roots(C.c, R.r);
  return R;
}

// Seeded solve: Newton iteration on the MONIC quintic (the caller divides the coefficients by c5), four independent
// chains at once, started from predictions of the roots (centre_seeds() in twk_contour.cuh).  Roots of a polynomial are
// continuous in its coefficients, so ghosts can be followed like real images.  The FIFTH root -- the one of largest
// modulus, which centre_seeds() orders last -- is not iterated: it follows from Vieta's sum, r4 = -c4 - (r0+r1+r2+r3).
// Stop rule per root: Newton converges quadratically, |dx_{n+1}| ~ K |dx_n|^2 with K ~ |dx_n| / |dx_{n-1}|^2, so
// the step AFTER the one just taken would be ~ |dx_n|^3 / |dx_{n-1}|^2; once that is below 1e-13 |r| (three orders
// inside the 1e-10 position bar) the root is converged and the confirming evaluation is skipped.  The rule compares
// orders of magnitude and runs on integer magnitude keys (mag_key).  From the third sweep on the residual is also
// compared with the rounding floor of its own evaluation (ill-conditioned roots next to a caustic stall there).
// Verification: the product of the five roots = -c0 (relative 1e-9; catches two chains on one root), and, once all
// five are iterated, their sum = -c4.
// Recovery (at most once per solve): when the product does not verify, or a chain has not converged after
// TWK_RECOVER_AT sweeps, chain 4 is iterated like the others for three sweeps; then the three or four good distinct roots
// fix the others through Vieta's formulas (sum = -c4, product = -c0: one missing root directly, two as the roots of a
// quadratic -- which is also the fast way through a nearly double root, where Newton converges only linearly); these are
// polished by the same Newton sweeps and verified again.
// Returns 0 when that fails too; the caller then falls back to the cold solver quintic_roots().
// r[] holds the seeds on entry and the roots on exit.
// Two converged chains are the same root when they agree to 1e-6 of their size (RELATIVE: next to a planet of
// q = 1e-9 two distinct roots can be 1e-9 apart in absolute terms while the other roots are of order one).
constexpr double kDupRel2 = 1e-12;
#ifndef TWK_RECOVER_AT
#define TWK_RECOVER_AT 4   // sweeps before chains that have not converged are replaced through Vieta's formulas
#endif

struct SeededState {
  cd r[5];
  unsigned done;
  int ok;
};
// Recovery step of the seeded solve (see above), out of line.  Returns ok = 0 when fewer than three good roots are
// left; otherwise the replaced roots are in r[] with their done bits cleared.
TWK_NOINLINE SeededState seeded_recover(cd c0, cd c5, cd tot, SeededState S) {
  TWK_COUNT(recovery);
  cd (&r)[5] = S.r;
  // good = converged and not a duplicate of an earlier good root
  unsigned good = S.done;
#pragma unroll
  for (int a = 0; a < 5; ++a)
#pragma unroll
    for (int b = a + 1; b < 5; ++b)
      if ((good >> a & 1u) && (good >> b & 1u) && norm2(r[a] - r[b]) <= kDupRel2 * (norm2(r[a]) + norm2(r[b])))
        good &= ~(1u << b);
  int ng = 0;
#pragma unroll
  for (int k = 0; k < 5; ++k) ng += (good >> k) & 1u;
  S.ok = (ng == 3 || ng == 4);
  if (!S.ok) return S;
  cd sum = mk(0.0, 0.0), prod = mk(1.0, 0.0);
#pragma unroll
  for (int k = 0; k < 5; ++k)
    if (good >> k & 1u) {
      sum = sum + r[k];
      prod = prod * r[k];
    }
  cd x1 = tot - sum, x2 = x1;
  if (ng == 3) {   // x^2 - S x + P = 0 with S = tot - sum, P = (-c0/c5) / prod
    const cd Ssum = x1;
    const cd P = -cdiv(c0, c5 * prod);
    cd sq = csqrt_(Ssum * Ssum - 4.0 * P);
    if (dotp(Ssum, sq) < 0.0) sq = -sq;
    x1 = 0.5 * (Ssum + sq);
    x2 = (norm2(x1) > 0.0) ? cdiv(P, x1) : x1;
  }
  bool first = true;
#pragma unroll
  for (int k = 0; k < 5; ++k)
    if (!(good >> k & 1u)) {
      r[k] = first ? x1 : x2;
      first = false;
    }
  S.done = good;
  return S;
}

// Magnitude key of a complex number: 2^16 (log2(|Re| + |Im|) + 1023), piecewise linear in the mantissa -- the high
// word of the 1-norm.  The stop rule compares orders of magnitude; it runs on these keys in the integer ALU instead of
// spending FP64 multiplications on it.  NaN gives the largest key (never "converged"), zero gives 0.
TWK_HD int mag_key(cd v) {
#ifdef __CUDA_ARCH__
  return (int)((unsigned)__double2hiint(abs1(v)) >> 4);   // (unsigned: a NaN of either sign is the largest key)
#else
  return 0;
#endif
}
TWK_HD int mag_key1(double v) {   // key of a non-negative (or NaN) real
#ifdef __CUDA_ARCH__
  return (int)((unsigned)__double2hiint(v) >> 4);
#else
  return 0;
#endif
}
constexpr int kKeyOne = 1023 << 16;                  // key of 1.0
constexpr int kKeyStop = (0x3d3c2000 >> 4) - kKeyOne;   // 2^16 log2(TWK_STOP_FACTOR * eps) = 2^16 log2(1e-13)
constexpr int kKeyMargin = 1 << 16;                  // the piecewise-linear log2 (< 0.09 per key): a factor 2 on |dx|^3 covers it

// Horner for p and p' of the MONIC quintic (c[5] is not read): the first two steps are additions
TWK_HD void horner_pd(const cd (&c)[6], cd x, cd& p, cd& d) {
  p = mk(x.x + c[4].x, x.y + c[4].y);
  d = mk(x.x + p.x, x.y + p.y);
  p = cfma(p, x, c[3]);
#pragma unroll
  for (int i = 2; i >= 0; --i) {
    d = cfma(d, x, p);
    p = cfma(p, x, c[i]);
  }
}
// One Newton step x <- x - p / p'; returns the magnitude key of the step.  p' = 0 needs no branch: the reciprocal of 0
// is an infinity whose refinement is NaN, the root becomes NaN, its key the largest there is, and a chain that never
// "converges" is what the Vieta recovery replaces.
TWK_HD int newton_move(cd p, cd d, cd& x) {
  const double inv = rcp1(norm2(d));
  const cd num = mk(fma(p.x, d.x, p.y * d.y), fma(p.y, d.x, -(p.x * d.y)));   // p conj(p'):  dx = num / |p'|^2
  x = mk(fma(-num.x, inv, x.x), fma(-num.y, inv, x.y));
  return mag_key1(abs1(num) * inv);   // |dx|_1 = (|Re num| + |Im num|) / |p'|^2
}
// stop rule: |dx|^3 <= 1e-13 |x| |dx_prev|^2 on magnitude keys (kprev = 0: no previous step, only dx = 0 passes)
TWK_HD bool newton_converged(int ks, int kprev, cd x) { return 3 * ks + kKeyMargin <= kKeyStop + mag_key(x) + 2 * kprev; }

// The step of the later sweeps (one root at a time): also compares the residual with the rounding floor of its own
// evaluation.  Returns true when the root is converged; prev = key of the previous |dx|.
TWK_HD bool newton_step_floor(const cd (&c)[6], cd& x, int& prev) {
  TWK_COUNT(newton_eval);
  cd p, d;
  horner_pd(c, x, p, d);
  {
    const double ax = abs1(x);
    double err = 1.0;
#pragma unroll
    for (int i = 4; i >= 0; --i) err = fma(err, ax, abs1(c[i]));
    if (abs1(p) <= 2.0 * kEps * err) return true;   // at the rounding floor
  }
  const int ks = newton_move(p, d, x);
  const bool conv = newton_converged(ks, prev, x);
  prev = ks;
  return conv;
}

// Returns 0 = failed (use the cold solver), 1 = solved, 2 = solved after the Vieta recovery.
TWK_HD int quintic_roots_seeded(const cd (&c)[6], cd (&r)[5], bool check_product) {
  int prev[5];
#pragma unroll
  for (int k = 0; k < 5; ++k) prev[k] = 0;
  const cd tot = -c[4];               // sum of the five roots (monic coefficients)
  unsigned done = 0;
  // sweeps 0 and 1: every root needs them (the stop rule wants two steps), so the four chains run unconditionally and
  // interleave (instruction-level parallelism); a step on an already converged root is harmless.  A rolled loop of two
  // sweeps (one copy of the four interleaved chains keeps the hot loop inside the instruction cache), no branch inside;
  // the stop rule is evaluated once after it, from the keys of the two steps
  int kfirst[4];   // key of the first step of each chain
#pragma unroll
  for (int k = 0; k < 4; ++k) kfirst[k] = 0;
#pragma unroll 1
  for (int it = 0; it < 2; ++it) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      cd p, d;
      horner_pd(c, r[k], p, d);
      kfirst[k] = prev[k];
      prev[k] = newton_move(p, d, r[k]);
    }
  }
#pragma unroll
  for (int k = 0; k < 4; ++k) done |= newton_converged(prev[k], kfirst[k], r[k]) ? (1u << k) : 0u;
  // The FIFTH root is not iterated: it follows from Vieta's sum, r4 = -c4 - (r0 + r1 + r2 + r3).  centre_seeds() puts the
  // root of largest modulus last, so the rounding of the sum (a few ulp of the LARGEST root) is a relative error of
  // a few ulp of r4 itself; the product of the five roots then verifies the solve.  v5 = that short cut is still on
  // (bit 4 of `done` is preset); it is dropped -- and chain 4 iterated from its seed like the others -- as soon as
  // something does not converge or verify.
  bool v5 = true;
  done |= 16u;
  int rec_at = TWK_RECOVER_AT;
  bool recovered = false;
  for (int it = 2; it < 24; ++it) {
    if (v5 && done != 31u && it >= rec_at) {   // a chain is slow: give the recovery all five chains to choose from
      v5 = false;
      done &= 15u;
      rec_at = it + 3;
    }
    if (done == 31u || (it >= rec_at && !recovered)) {
      if (done == 31u) {
        if (v5) r[4] = tot - ((r[0] + r[1]) + (r[2] + r[3]));
        // verification by Vieta: the product of the roots (relative) catches two chains on one root -- also where the sum
        // is blind (a symmetric sample: equal masses, zeta = 0; roots 1e-9 of the scale apart next to a tiny planet; a
        // root that has run off towards infinity) -- and, when all five were iterated, the sum (on the scale of the largest)
        bool ok = true;
        if (!v5) {
          const double scale = abs1(r[0]) + abs1(r[1]) + abs1(r[2]) + abs1(r[3]) + abs1(r[4]);
          ok = abs1((r[0] + r[1]) + (r[2] + r[3]) + r[4] - tot) <= 1e-9 * scale;
        }
        {
          const cd prod = ((r[0] * r[1]) * (r[2] * r[3])) * r[4];
          ok = ok && abs1(prod + c[0]) <= 1e-9 * abs1(c[0]);                 // prod = -c0 (monic)
        }
        (void)check_product;
        if (ok) return recovered ? 2 : 1;
      }
      if (recovered) break;
      recovered = true;
      SeededState S;
#pragma unroll
      for (int k = 0; k < 5; ++k) S.r[k] = r[k];
      S.done = v5 ? (done & 15u) : done;   // (a Vieta-derived r4 is not evidence)
      v5 = false;
      S.ok = 0;
      S = seeded_recover(c[0], mk(1.0, 0.0), tot, S);
      if (!S.ok) break;
#pragma unroll
      for (int k = 0; k < 5; ++k)
        if (!(S.done >> k & 1u)) {
          r[k] = S.r[k];
          prev[k] = 0;
        }
      done = S.done;
    }
    // one step of every unfinished root; the root is moved through scalars (no dynamic indexing: r[] and prev[] stay
    // in registers), one copy of the step's code
#pragma unroll 1
    for (int k = 0; k < 5; ++k) {
      if (done & (1u << k)) continue;
      cd x = r[0];
      int pv = prev[0];
#pragma unroll
      for (int j = 1; j < 5; ++j)
        if (j == k) { x = r[j]; pv = prev[j]; }
      const bool cv = newton_step_floor(c, x, pv);
#pragma unroll
      for (int j = 0; j < 5; ++j)
        if (j == k) { r[j] = x; prev[j] = pv; }
      if (cv) done |= 1u << k;
    }
  }
  TWK_COUNT(fail_iter);
  return 0;
}

}  // namespace twk
