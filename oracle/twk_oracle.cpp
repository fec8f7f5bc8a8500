// twk_oracle.cpp -- TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, obviously-correct CPU statement of what the hot path computes: finite-source binary-lens
// magnification by contour integration, written from /root/reference/PAPER.md ("P:<line>" below) and the
// readings listed in DESIGN.md.  It shares NO code with the CUDA path (own coefficient builder, own root
// finder -- Durand-Kerner, not the product's Laguerre --, own linker, own integrator, own samplers).  Only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it; the
// product never does.
//
// Every routine is a template on the real type: `double` is the precision the method computes in (the
// default face, the one timed as cpu_baseline), `long double` (x87 80-bit here) is the extended-precision
// twin used to pin coefficient accuracy and classification.  prec = 0 -> double, 1 -> long double.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): coefficients vs mpmath elimination of Eq.(1); roots vs
// Vieta/backward error; sum of residuals = 0; ghost 2-cycle geometry; 3-or-5 images, parity sum -1
// (P:155-159); generalised point-source magnification sum = 1; z' and z'^z'' vs finite differences of tracked
// images; single-lens limits (Paczynski point source, uniform-disk closed forms); large-rho limit;
// mass-swap / reflection symmetries; brute-force ray shooting on tiny inputs; the Fig.1 / Fig.2 worked
// examples.  tests/test_oracle_errors.py: the crossing piece Eq.(11) and the estimate Eq.(18)
// against the closed forms of a fold model (creation and annihilation separately) and against fine integrations of
// the same interval on real lenses; Eq.(17) term by term against 50-digit mpmath image tracks; the estimate's honesty
// interval by interval; the sampler against hand-computed quantiles; the parity repair against Eq.(7).
// Unpinned: adaptive-mode *sample positions* on real sources (only mu, n and status are compared); slope-detector
// decisions at the default gate (it never fires).

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

template <class R> using Cx = std::complex<R>;

template <class R> inline R wedge(const Cx<R>& a, const Cx<R>& b) { return a.real() * b.imag() - a.imag() * b.real(); }
template <class R> inline R dot(const Cx<R>& a, const Cx<R>& b) { return a.real() * b.real() + a.imag() * b.imag(); }

// ---------------------------------------------------------------------------------------------------------
// O1. lens geometry, Eq.(2)
// ---------------------------------------------------------------------------------------------------------
template <class R> struct Lens {
  R s, q, m1, m2, z1, z2;
};
template <class R> Lens<R> make_lens(double s_, double q_) {
  Lens<R> L;
  L.s = (R)s_;
  L.q = (R)q_;
  L.m1 = R(1) / (R(1) + L.q);
  L.m2 = L.q / (R(1) + L.q);
  L.z1 = -L.q * L.s / (R(1) + L.q);
  L.z2 = L.s / (R(1) + L.q);
  return L;
}

// ---------------------------------------------------------------------------------------------------------
// O2. polynomial coefficients in the planet frame (planet at 0, primary at -s), Eq.(6), as printed.
// ---------------------------------------------------------------------------------------------------------
template <class R> void coeffs_eq6(const Cx<R>& y, R s, R m2, Cx<R> c[6]) {
  const Cx<R> I(0, 1);
  const Cx<R> yb = std::conj(y);
  const Cx<R> vc = yb + s;            // v_c = ybar + s
  const Cx<R> vp = R(1) + s * yb;     // v_p = 1 + s ybar
  const R Iy = y.imag();
  c[5] = -yb * vc;
  c[4] = (yb * y - R(1) - R(2) * s * yb) * vc + m2 * s;
  c[3] = (R(2) * y - s) * (vp * vc + R(2) * Iy * I - m2 * s) + R(4) * (m2 * s - y) * Iy * I;
  c[2] = vp.real() * vp.real() * vc.real() + Iy * vp.real() * (R(1) - s * y).real() * I +
         s * Iy * Iy * (R(2) + s * vc) + m2 * s * (R(2) * yb * (y - s) - (R(1) - s * y));
  c[1] = m2 * s * ((s + R(2) * y) * vp + s * (R(2) * s * Iy * I - m2));
  c[0] = s * s * m2 * m2 * y;
}

// The conventional form Eq.(4), with the OCR repair of c3 ("+ s [y + 2 ybar (ybar y - m2)]", DESIGN.md
// reading E-1).  NOT on any path: kept only as the foil of the cancellation test.
template <class R> void coeffs_eq4(const Cx<R>& y, R s, R m1, R m2, Cx<R> c[6]) {
  const Cx<R> yb = std::conj(y);
  c[5] = -yb * (yb + s);
  c[4] = yb * (yb * (R(-2) * s + y) - R(1)) + s * (yb * (R(-2) * s + y) - m1);
  c[3] = R(2) * yb * y - s * s * s * yb + s * s * (yb * (R(2) * y - yb) - m1) + s * (y + R(2) * yb * (yb * y - m2));
  c[2] = y * (R(1) + s * s * s * yb) + s * (m1 + R(2) * y * yb * (R(1) + m2)) +
         s * s * (yb * (m1 - m2) + y * (R(1) + m2 + yb * yb));
  c[1] = m2 * s * (s * (m1 + y * (R(2) * yb + s)) + R(2) * y);
  c[0] = s * s * m2 * m2 * y;
}

// ---------------------------------------------------------------------------------------------------------
// O3. quintic roots: Durand-Kerner (Weierstrass) simultaneous iteration + Newton polish on the undeflated
// polynomial.  Textbook; deliberately a different algorithm from the product's solver.
// ---------------------------------------------------------------------------------------------------------
template <class R> inline Cx<R> horner(const Cx<R> c[6], const Cx<R>& x) {
  Cx<R> p = c[5];
  for (int i = 4; i >= 0; --i) p = p * x + c[i];
  return p;
}
template <class R> inline void horner2(const Cx<R> c[6], const Cx<R>& x, Cx<R>& p, Cx<R>& dp) {
  p = c[5];
  dp = Cx<R>(0, 0);
  for (int i = 4; i >= 0; --i) {
    dp = dp * x + p;
    p = p * x + c[i];
  }
}

template <class R> int quintic_roots_dk(const Cx<R> c[6], Cx<R> r[5]) {
  const R eps = std::numeric_limits<R>::epsilon();
  Cx<R> b[6];
  for (int i = 0; i < 6; ++i) b[i] = c[i] / c[5];
  // Fujiwara bound on the root moduli
  R rad = 0;
  for (int k = 1; k <= 5; ++k) {
    R t = std::pow(std::abs(b[5 - k]) * (k == 5 ? R(0.5) : R(1)), R(1) / R(k));
    rad = std::max(rad, t);
  }
  rad *= R(2);
  if (!(rad > 0)) rad = 1;
  const Cx<R> ctr = -b[4] / R(5);
  const R r0 = R(0.5) * rad + std::abs(ctr) * R(0.1) + std::numeric_limits<R>::min();
  const R twopi = R(2) * std::acos(R(-1));
  for (int k = 0; k < 5; ++k) r[k] = ctr + std::polar(r0, twopi * R(k) / R(5) + R(0.4));
  int sweep = 0, stalled = 0;
  R best = std::numeric_limits<R>::infinity();
  for (; sweep < 2000; ++sweep) {
    R maxrel = 0;
    for (int k = 0; k < 5; ++k) {
      Cx<R> num = horner(b, r[k]);
      Cx<R> den(1, 0);
      for (int j = 0; j < 5; ++j)
        if (j != k) den *= (r[k] - r[j]);
      if (den == Cx<R>(0, 0)) den = Cx<R>(eps, eps);
      Cx<R> d = num / den;
      r[k] -= d;
      maxrel = std::max(maxrel, std::abs(d) / std::max(std::abs(r[k]), std::numeric_limits<R>::min()));
    }
    if (maxrel < R(2) * eps) break;
    // ill-conditioned clusters never reach 2 eps: stop once the update size has stopped shrinking
    if (maxrel < R(0.5) * best) { best = maxrel; stalled = 0; } else if (maxrel < R(1e-6) && ++stalled >= 8) break;
  }
  // Newton polish on the full polynomial (3 steps; a step is taken only if it does not increase |P|)
  for (int k = 0; k < 5; ++k) {
    for (int it = 0; it < 3; ++it) {
      Cx<R> p, dp;
      horner2(c, r[k], p, dp);
      if (dp == Cx<R>(0, 0)) break;
      Cx<R> x1 = r[k] - p / dp;
      if (std::abs(horner(c, x1)) <= std::abs(p)) r[k] = x1; else break;
    }
  }
  return sweep;
}

// ---------------------------------------------------------------------------------------------------------
// O1 + O4 + O5: one boundary point source -> five roots, residuals, Jacobians, classification, z', z'^z''.
// ---------------------------------------------------------------------------------------------------------
template <class R> struct Sample {
  R theta;
  Cx<R> zeta, dzeta;  // boundary point and d zeta / d theta = i rho e^{i theta}
  Cx<R> c[6];         // Eq.(6) coefficients
  Cx<R> z[5];         // all five roots, CM frame
  Cx<R> Res[5];       // Eq.(12) residuals
  R J[5];             // Eq.(7)
  int kind[5];        // 0 ghost, +1 / -1 real image parity
  Cx<R> zp[5];        // z' = dz/dtheta   (Eq.10, corrected: conj on f')
  R w[5];             // z' ^ z''         (Eq.10, corrected: divided by J)
  int nreal;
  int repaired;       // parity repair fired (reading G-5)
  int slope;          // a real pair of this sample was re-judged as ghosts by the slope detector
  int guard;          // the sample sat on a lens and was moved off it (reading B-1)
  int sweeps;
};

template <class R>
void point_solve(const Lens<R>& L, const Cx<R>& zc, R rho, R theta, Sample<R>& S) {
  S.theta = theta;
  const Cx<R> e(std::cos(theta), std::sin(theta));
  S.zeta = zc + rho * e;
  S.dzeta = Cx<R>(0, 1) * rho * e;
  Cx<R> y = S.zeta - L.z2;
  // B-1: a boundary point ON a lens (conj(y) = 0 or conj(y) = -s) makes c5 = 0: one root escapes to
  // infinity and one sits on the pole of f.  The magnification is continuous there, so a point closer to a lens than
  // 1e-14 s -- the rounding of zeta itself -- is moved to that distance (along the lens axis); status bit 16.
  S.guard = 0;
  const R dmin = R(1e-14) * L.s;
  if (std::abs(y) < dmin) { y = Cx<R>(dmin, 0); S.guard = 1; }
  if (std::abs(y + L.s) < dmin) { y = Cx<R>(-L.s + dmin, 0); S.guard = 1; }
  coeffs_eq6(y, L.s, L.m2, S.c);
  Cx<R> eta[5];
  S.sweeps = quintic_roots_dk(S.c, eta);
  Cx<R> fpp[5], fp[5];
  for (int k = 0; k < 5; ++k) {
    // planet frame: z2 - z = -eta, z1 - z = -s - eta  (Eq.12 and Eq.7 are frame invariant)
    const Cx<R> a = R(1) / (-L.s - eta[k]);
    const Cx<R> b = R(1) / (-eta[k]);
    const Cx<R> f = L.m1 * a + L.m2 * b;                           // Eq.(7)
    fp[k] = L.m1 * a * a + L.m2 * b * b;                           // f'
    fpp[k] = R(2) * (L.m1 * a * a * a + L.m2 * b * b * b);         // f''
    S.Res[k] = y - eta[k] - std::conj(f);                          // Eq.(12)
    S.J[k] = R(1) - std::norm(fp[k]);                              // Eq.(7)
    S.z[k] = eta[k] + L.z2;
  }
  // residual detector, P:205-249, 2-cycle reading (G-1): the two largest-|R| roots a,b are a ghost
  // pair iff R_a = z_b - z_a and R_b = z_a - z_b ("a pair of ghost images with opposite residuals").
  int ia = 0, ib = 1;
  {
    int idx[5] = {0, 1, 2, 3, 4};
    std::sort(idx, idx + 5, [&](int u, int v) { return std::abs(S.Res[u]) > std::abs(S.Res[v]); });
    ia = idx[0];
    ib = idx[1];
  }
  const Cx<R> dab = eta[ib] - eta[ia];
  const bool ghost = std::abs(S.Res[ia] - dab) < std::abs(S.Res[ia]) && std::abs(S.Res[ib] + dab) < std::abs(S.Res[ib]);
  S.nreal = 0;
  int npos = 0;
  for (int k = 0; k < 5; ++k) {
    if (ghost && (k == ia || k == ib)) { S.kind[k] = 0; continue; }
    S.kind[k] = (S.J[k] > 0) ? +1 : -1;   // Eq.(7)
    S.nreal++;
    npos += (S.kind[k] > 0);
  }
  // parity sum must be -1: (1+,2-) or (2+,3-).  If rounding next to the critical curve broke it, flip
  // the smallest-|J| image of the over-represented parity (reading G-5).
  S.repaired = 0;
  S.slope = 0;
  const int want = (S.nreal - 1) / 2;
  while (npos != want) {
    int best = -1;
    for (int k = 0; k < 5; ++k) {
      if (S.kind[k] == 0) continue;
      if ((npos > want) != (S.kind[k] > 0)) continue;
      if (best < 0 || std::abs(S.J[k]) < std::abs(S.J[best])) best = k;
    }
    S.kind[best] = -S.kind[best];
    npos += S.kind[best];   // +1 if flipped to +, -1 if flipped to -
    S.repaired = 1;
  }
  for (int k = 0; k < 5; ++k) {
    // Eq.(10) with the two OCR repairs (E-2, E-3)
    S.zp[k] = (S.dzeta - std::conj(fp[k]) * std::conj(S.dzeta)) / S.J[k];
    S.w[k] = (rho * rho + (S.zp[k] * S.zp[k] * S.dzeta * fpp[k]).imag()) / S.J[k];
  }
}

const double kPi = 3.14159265358979323846264338327950288;
template <class R> R pi_v() { return std::acos(R(-1)); }

// ---------------------------------------------------------------------------------------------------------
// O6 + O7: one interval (theta_i -> theta_{i+1}): link, area piece, error piece.
// ---------------------------------------------------------------------------------------------------------
template <class R> struct Piece {
  R dA, err;
  int crossing;  // 0 none, +1 creation, -1 annihilation
  int bad;       // leftover images are not exactly one (+,-) pair on one side
  int slope;     // slope detector (reading G-4): the crossing's real pair (kp, km) is not perpendicular to
  int kp, km;    // the ghost pair of the 3-image sample next to it and must be re-judged as ghosts
  int nlinks;
  int linkL[5], linkR[5];  // root indices of the linked pairs (diagnostics / tests)
  // diagnostics for the pins (no effect on dA / err): the interval's error estimate term by term --
  // [0..3] Eq.(17) E1..E4 summed over the regular links, [4..6] Eq.(18) E1..E3 of the crossing, [7] the crossing's
  // Eq.(11) correction as it entered dA (signed)
  R terms[8];
};

template <class R>
void eval_interval(const Sample<R>& A, const Sample<R>& B, R dth, Piece<R>& P, R slope_gate2 = R(0), R slope_cos2 = R(0.5)) {
  P.dA = 0;
  P.err = 0;
  P.crossing = 0;
  P.bad = 0;
  P.slope = 0;
  P.kp = P.km = -1;
  P.nlinks = 0;
  for (int k = 0; k < 8; ++k) P.terms[k] = 0;
  int leftA[5], leftB[5], nLA = 0, nLB = 0;
  for (int par = +1; par >= -1; par -= 2) {
    int ia[5], ib[5], na = 0, nb = 0;
    for (int k = 0; k < 5; ++k) {
      if (A.kind[k] == par) ia[na++] = k;
      if (B.kind[k] == par) ib[nb++] = k;
    }
    // injective maps of the smaller set into the larger one; keep the one of minimum total distance
    const bool a_small = na <= nb;
    const int* sm = a_small ? ia : ib;
    const int* lg = a_small ? ib : ia;
    const int ns = a_small ? na : nb, nl = a_small ? nb : na;
    const Sample<R>& Ss = a_small ? A : B;
    const Sample<R>& Sl = a_small ? B : A;
    int perm[5] = {0, 1, 2, 3, 4}, bestp[5] = {0, 1, 2, 3, 4};
    R best = std::numeric_limits<R>::infinity();
    do {
      R cost = 0;
      for (int j = 0; j < ns; ++j) cost += std::abs(Ss.z[sm[j]] - Sl.z[lg[perm[j]]]);
      if (cost < best) {
        best = cost;
        std::copy(perm, perm + 5, bestp);
      }
    } while (std::next_permutation(perm, perm + nl));
    for (int j = 0; j < ns; ++j) {
      const int ka = a_small ? sm[j] : lg[bestp[j]];
      const int kb = a_small ? lg[bestp[j]] : sm[j];
      P.linkL[P.nlinks] = ka;
      P.linkR[P.nlinks] = kb;
      P.nlinks++;
      const Cx<R> dz = B.z[kb] - A.z[ka];
      const R trap = R(0.5) * wedge(A.z[ka], dz);                                    // Eq.(9)
      const R p1 = (A.w[ka] + B.w[kb]) * dth * dth * dth / R(24);                    // Eq.(10) dA^(p1)
      const R p2 = wedge(dz, B.zp[kb] - A.zp[ka]) * dth / R(12);                     // Eq.(10) dA^(p2)
      const R dAp = R(0.5) * (p1 + p2);
      P.dA += R(par) * (trap + dAp);
      const R E1 = std::abs(A.w[ka] - B.w[kb]) * dth * dth * dth / R(48);            // Eq.(17)
      const R E2 = R(1.5) * std::abs(dAp * (std::norm(dz) / (dth * dth * std::abs(dot(A.zp[ka], B.zp[kb]))) - R(1)));
      const R E3 = R(0.1) * std::abs(dAp) * dth * dth;
      const R E4 = std::abs(p1 - p2);
      P.err += E1 + E2 + E3 + E4;
      P.terms[0] += E1; P.terms[1] += E2; P.terms[2] += E3; P.terms[3] += E4;
    }
    for (int j = ns; j < nl; ++j) {
      if (a_small) leftB[nLB++] = lg[bestp[j]]; else leftA[nLA++] = lg[bestp[j]];
    }
  }
  if (nLA == 0 && nLB == 0) return;
  // the extra real pair on the 5-image side connects to itself
  const bool creation = (nLA == 0 && nLB == 2 && B.kind[leftB[0]] * B.kind[leftB[1]] == -1);
  const bool annihil = (nLB == 0 && nLA == 2 && A.kind[leftA[0]] * A.kind[leftA[1]] == -1);
  if (!creation && !annihil) {
    P.bad = 1;
    P.err = std::numeric_limits<R>::infinity();
    return;
  }
  const Sample<R>& S = creation ? B : A;
  const int* lf = creation ? leftB : leftA;
  const int kp = (S.kind[lf[0]] > 0) ? lf[0] : lf[1];
  const int km = (S.kind[lf[0]] > 0) ? lf[1] : lf[0];
  const Cx<R> zpl = S.z[kp], zmi = S.z[km];
  const Cx<R> d = zpl - zmi;
  {
    // Slope detector, P:251-268 (reading G-4): next to the critical curve the real pair (5-image sample) and the
    // ghost pair (3-image sample) are perpendicular.  Applied only when both pairs are closer than the gate
    // ("works only for the point sources near caustics"); |cos| >= cos 45 deg = the pair is misjudged.
    const Sample<R>& G = creation ? A : B;
    int g[2], ng = 0;
    for (int k = 0; k < 5 && ng < 2; ++k)
      if (G.kind[k] == 0) g[ng++] = k;
    if (ng == 2) {
      const Cx<R> dg = G.z[g[0]] - G.z[g[1]];
      const R nr = std::norm(d), ngg = std::norm(dg), c = dot(d, dg);
      if (nr < slope_gate2 && ngg < slope_gate2 && c * c >= slope_cos2 * nr * ngg) {
        P.slope = 1;
        P.kp = kp;
        P.km = km;
      }
    }
  }
  const R sq = std::sqrt(std::abs(dot(S.zp[kp], S.zp[km])));
  const R dtt = std::abs(d) / sq;                                                    // Eq.(11) tilde Delta theta
  const R corr = (S.w[kp] - S.w[km]) * dtt * dtt * dtt / R(24);                      // Eq.(11)
  // Eq.(11) enters as printed in BOTH directions (reading S-2): the + track is followed with
  // increasing theta, the - track against it, so the pair's path is z- -> (critical curve) -> z+ at a creation and
  // z+ -> z- at an annihilation; only the closing chord changes direction.  For the fold model
  // z+- = zc + a d t ^ +- b sqrt(d) n ^ (d = |theta - theta_c|) the printed correction equals the area between that
  // path and its chord exactly, with the same sign in both cases (tests/test_oracle_errors.py, fold model).
  const R dAp = corr;
  R chord, E2;
  if (creation) {   // path z- -> z+
    chord = R(0.5) * wedge(zmi, d);
    E2 = R(1.5) * std::abs(dot(d, S.zp[kp] - S.zp[km]) - R(2) * std::abs(d) * sq) * dtt;   // Eq.(18), E-5; '-' P:302
  } else {          // path z+ -> z-
    chord = R(0.5) * wedge(zpl, -d);
    E2 = R(1.5) * std::abs(dot(d, S.zp[kp] - S.zp[km]) + R(2) * std::abs(d) * sq) * dtt;   // '+' P:302
  }
  P.crossing = creation ? +1 : -1;
  P.dA += chord + dAp;
  const R E1 = std::abs(S.w[kp] + S.w[km]) * dtt * dtt * dtt / R(48);                // Eq.(18)
  const R E3 = R(0.1) * std::abs(dAp) * dth * dth;
  P.err += E1 + E2 + E3;
  P.terms[4] = E1; P.terms[5] = E2; P.terms[6] = E3; P.terms[7] = dAp;
}


// ---------------------------------------------------------------------------------------------------------
// L-4 guard (an EXTENSION of the paper's estimate, off by default; reading L-4).  The estimates of Eq.(17)
// see an interval through its end points only: a boundary that dips into a caustic and out again BETWEEN two adjacent
// samples (both with 3 images) leaves no trace in them.  The ghost pair does: next to a fold its separation squared
// D = |z_a - z_b|^2 is proportional to the distance of the boundary point from the caustic, so along the boundary it
// follows a parabola in theta that reaches zero where the boundary touches the caustic and would turn negative inside,
// where the pair is real with the same separation law.  For the interval (A, B), D is fitted through (A-, A, B) and
// through (A, B, B+) (neighbours with 3 images only); a convex fit whose vertex lies inside the interval at a negative
// value D* means a hidden pair of crossings 2 sqrt(-D*/C) apart (C = the fit's curvature), whose images enclose the
// area  v (pi/2) (-D*) / sqrt(C)  (half an ellipse: pair separation sqrt(-D) across, v = speed of the pair's midpoint
// along the critical curve, taken from the ghost midpoints of A and B).  That area is added to the interval's error
// estimate, so the sampler refines there until the crossings are seen or the hidden area is negligible.
// dm, d, dp = theta_A - theta_A-, theta_B - theta_A, theta_B+ - theta_B  (> 0).
// ---------------------------------------------------------------------------------------------------------
template <class R>
bool ghost_pair(const Sample<R>& S, Cx<R>& sep, Cx<R>& mid) {
  if (S.nreal != 3) return false;
  int g[2], ng = 0;
  for (int k = 0; k < 5 && ng < 2; ++k)
    if (S.kind[k] == 0) g[ng++] = k;
  if (ng != 2) return false;
  sep = S.z[g[0]] - S.z[g[1]];
  mid = R(0.5) * (S.z[g[0]] + S.z[g[1]]);
  return true;
}

template <class R>
R hidden_crossing_term(const Sample<R>* Am, const Sample<R>& A, const Sample<R>& B, const Sample<R>* Bp, R dm, R d, R dp) {
  Cx<R> sA, mA, sB, mB, s3, m3;
  if (!ghost_pair(A, sA, mA) || !ghost_pair(B, sB, mB)) return R(0);
  const R DA = std::norm(sA), DB = std::norm(sB);
  const R v = std::abs(mB - mA) / d;
  R term = 0;
  for (int side = 0; side < 2; ++side) {
    const Sample<R>* T = side ? Bp : Am;
    if (!T || !ghost_pair(*T, s3, m3)) continue;
    // three points (x0,y0),(x1,y1),(x2,y2) in theta - theta_A, in increasing order
    const R x0 = side ? R(0) : -dm, x1 = side ? d : R(0), x2 = side ? d + dp : d;
    const R y0 = side ? DA : std::norm(s3), y1 = side ? DB : DA, y2 = side ? std::norm(s3) : DB;
    const R f01 = (y1 - y0) / (x1 - x0), f12 = (y2 - y1) / (x2 - x1);
    const R C = (f12 - f01) / (x2 - x0);
    if (!(C > 0)) continue;
    const R xs = R(0.5) * (x0 + x1) - f01 / (R(2) * C);
    if (!(xs > 0 && xs < d)) continue;
    const R ys = y0 + f01 * (xs - x0) + C * (xs - x0) * (xs - x1);
    if (!(ys < 0)) continue;
    term = std::max(term, v * R(0.5) * pi_v<R>() * (-ys) / std::sqrt(C));
  }
  return term;
}

// ---------------------------------------------------------------------------------------------------------
// Fixed-sampling face: theta_j = 2 pi j / N.
// ---------------------------------------------------------------------------------------------------------
template <class R>
void images_fixed_one(double s, double q, double rho_, double zre, double zim, int N, double* out_z, int8_t* out_kind,
                      int8_t* out_count, double* out_mu, double* out_err, int32_t* out_ncross, double* out_piece) {
  const Lens<R> L = make_lens<R>(s, q);
  const R rho = (R)rho_;
  const Cx<R> zc((R)zre, (R)zim);
  std::vector<Sample<R>> S(N);
  const R twopi = R(2) * pi_v<R>();
  for (int j = 0; j < N; ++j) {
    point_solve(L, zc, rho, twopi * R(j) / R(N), S[j]);
    for (int k = 0; k < 5; ++k) {
      if (out_z) {
        out_z[(size_t(j) * 5 + k) * 2 + 0] = (double)S[j].z[k].real();
        out_z[(size_t(j) * 5 + k) * 2 + 1] = (double)S[j].z[k].imag();
      }
      if (out_kind) out_kind[size_t(j) * 5 + k] = (int8_t)S[j].kind[k];
    }
    if (out_count) out_count[j] = (int8_t)S[j].nreal;
  }
  R A = 0, E = 0;
  int ncross = 0;
  const R dth = twopi / R(N);
  for (int j = 0; j < N; ++j) {
    Piece<R> P;
    eval_interval(S[j], S[(j + 1) % N], dth, P);
    A += P.dA;
    E += P.err;
    ncross += (P.crossing != 0);
    if (out_piece) {
      out_piece[2 * j] = (double)P.dA;
      out_piece[2 * j + 1] = (double)P.err;
    }
  }
  if (out_mu) *out_mu = (double)(A / (pi_v<R>() * rho * rho));
  if (out_err) *out_err = (double)(E / std::abs(A));
  if (out_ncross) *out_ncross = ncross;
}

// ---------------------------------------------------------------------------------------------------------
// Adaptive face.  mode 0: the paper's sampler (readings A-1..A-6).
//                 mode 1: the oracle's own converged reference (bisection of the worst intervals, O8).
// ---------------------------------------------------------------------------------------------------------
struct AdaptOpt {
  int samples_per_iter, initial_samples, max_samples, subtract_avg_tol;
  double slope_gate;   // slope detector proximity gate (0 = off)
  double slope_cos;    // largest |cos| still counted as perpendicular (cos 45 deg: reading G-4)
  int hidden_guard;    // L-4 guard (extension, default 0)
};

template <class R> struct Contour {
  Lens<R> L;
  Cx<R> zc;
  R rho;
  std::vector<Sample<R>> S;   // sorted by theta
  std::vector<Piece<R>> P;    // P[i] = interval (S[i], S[i+1 mod n])
  R twopi;
  R gate2 = R(0);             // square of the slope detector's gate
  R cos2 = R(0.5);            // square of the largest |cos| counted as perpendicular
  int guard = 0;              // L-4 guard: add the hidden-crossing term to the interval estimates
  void init(int n0) {
    S.resize(n0);
    for (int j = 0; j < n0; ++j) point_solve(L, zc, rho, twopi * R(j) / R(n0), S[j]);
    P.resize(n0);
    for (int j = 0; j < n0; ++j) eval(j);
    slope_repair();
  }
  // Slope detector: "When the slope detector finds that the perpendicular condition is not satisfied, nearby
  // image pairs are checked until the slope jump position is found or reaches the end of the image piece."  Rounds:
  // re-judge the pairs flagged by a creation (sample to the right of the interval), then those flagged by an
  // annihilation (sample to the left, if it still has five images), evaluate every interval again; repeat until no
  // crossing is flagged.  A piece whose pairs are never perpendicular disappears pair by pair ("the whole area piece
  // shall be deleted").
  static void demote(Sample<R>& s, int kp, int km) {
    s.kind[kp] = 0;
    s.kind[km] = 0;
    s.nreal = 3;
    s.slope = 1;
  }
  void slope_repair() {
    for (;;) {
      const int n = (int)S.size();
      std::vector<int> flagged;
      for (int i = 0; i < n; ++i)
        if (P[i].slope) flagged.push_back(i);
      if (flagged.empty()) return;
      for (int i : flagged)
        if (P[i].crossing > 0) demote(S[(i + 1) % n], P[i].kp, P[i].km);
      for (int i : flagged)
        if (P[i].crossing < 0 && S[i].nreal == 5) demote(S[i], P[i].kp, P[i].km);
      for (int i = 0; i < n; ++i) eval(i);
    }
  }
  R dtheta(int i) const {
    const int n = (int)S.size();
    return (i + 1 < n) ? S[i + 1].theta - S[i].theta : twopi - S[i].theta + S[0].theta;
  }
  void eval(int i) {
    const int n = (int)S.size();
    eval_interval(S[i], S[(i + 1) % n], dtheta(i), P[i], gate2, cos2);
    if (guard && n >= 4 && !P[i].bad && P[i].crossing == 0) {
      const int im = (i + n - 1) % n, ib = (i + 1) % n, ip = (i + 2) % n;
      P[i].err += hidden_crossing_term(&S[im], S[i], S[ib], &S[ip], dtheta(im), dtheta(i), dtheta(ib));
    }
  }
  // insert new angles (each strictly inside some interval), re-evaluate only the changed intervals
  void insert(std::vector<R> th) {
    std::sort(th.begin(), th.end());
    std::vector<Sample<R>> S2;
    std::vector<Piece<R>> P2;
    std::vector<char> dirty;
    const int n = (int)S.size();
    size_t t = 0;
    for (int i = 0; i < n; ++i) {
      S2.push_back(S[i]);
      P2.push_back(P[i]);
      dirty.push_back(0);
      const R hi = (i + 1 < n) ? S[i + 1].theta : twopi;
      while (t < th.size() && th[t] < hi) {
        if (th[t] > S2.back().theta) {
          Sample<R> ns;
          point_solve(L, zc, rho, th[t], ns);
          dirty.back() = 1;
          S2.push_back(ns);
          P2.push_back(Piece<R>());
          dirty.push_back(1);
        }
        ++t;
      }
    }
    S.swap(S2);
    P.swap(P2);
    for (size_t i = 0; i < S.size(); ++i)
      if (dirty[i]) eval((int)i);
    slope_repair();
  }
  void sums(R& A, R& E, int& nbad) const {
    A = 0;
    E = 0;
    nbad = 0;
    for (const auto& p : P) {
      A += p.dA;
      if (p.bad) nbad++; else E += p.err;
    }
  }
};

// ---------------------------------------------------------------------------------------------------------
// a8. One step of the paper's sampler (Fig.4): the per-interval errors are the sampling weights; the
// normalised cumulative error is inverted at K quantiles placed uniformly on the vertical axis, with linear
// interpolation inside the interval.  theta[] sorted, err[i] / bad[i] belong to the interval (theta_i, theta_{i+1})
// (cyclic, the last one closes at 2 pi + theta_0); tolA = tol * |A|.
//   A-4  quantile k sits at (k + 1/2) / K of the total weight: the only uniform placement for which K quantiles
//        give K NEW samples (Fig.4's caption: "generates eight new samples"); k / K and (k + 1) / K each put one
//        quantile on an existing sample.
//   A-5  "we subtract each error by the average tolerance": w_i = max(e_i - tolA / n, 0); an interval already
//        below its share gets no new sample.  If every weight vanishes the raw errors are used.
//   A-7  inconsistent intervals (oracle only) share half of the quantiles.
// Returns the new angles (those strictly inside their interval), in quantile order.
// ---------------------------------------------------------------------------------------------------------
template <class R>
std::vector<R> sampler_new_thetas(const std::vector<R>& theta, const std::vector<R>& err, const std::vector<char>& bad,
                                  R twopi, R tolA, int K, int subtract_avg_tol) {
  const int n = (int)theta.size();
  auto dtheta = [&](int i) { return (i + 1 < n) ? theta[i + 1] - theta[i] : twopi - theta[i] + theta[0]; };
  int nbad = 0;
  for (int i = 0; i < n; ++i) nbad += bad[i] ? 1 : 0;
  std::vector<R> wgt(n);
  const R avg = subtract_avg_tol ? tolA / R(n) : R(0);                              // P:306, A-5
  R W = 0;
  for (int i = 0; i < n; ++i) {
    wgt[i] = bad[i] ? R(0) : std::max(err[i] - avg, R(0));
    W += wgt[i];
  }
  if (nbad) {   // inconsistent intervals take half of the quantiles (reading A-7)
    const R wb = (W + tolA) / R(nbad);
    W = 0;
    for (int i = 0; i < n; ++i) {
      if (bad[i]) wgt[i] = wb;
      W += wgt[i];
    }
  }
  if (!(W > 0)) {
    W = 0;
    for (int i = 0; i < n; ++i) { wgt[i] = err[i]; W += wgt[i]; }
  }
  std::vector<R> cum(n + 1);
  cum[0] = 0;
  for (int i = 0; i < n; ++i) cum[i + 1] = cum[i] + wgt[i];
  std::vector<R> newth;
  for (int k = 0; k < K; ++k) {
    const R target = (R(k) + R(0.5)) / R(K) * cum[n];                               // quantiles, A-4
    int i = int(std::upper_bound(cum.begin(), cum.end(), target) - cum.begin()) - 1;
    i = std::min(std::max(i, 0), n - 1);
    while (i < n - 1 && !(wgt[i] > 0)) ++i;
    const R frac = wgt[i] > 0 ? (target - cum[i]) / wgt[i] : R(0.5);
    const R th = theta[i] + frac * dtheta(i);                                       // linear interpolation
    const R hi = (i + 1 < n) ? theta[i + 1] : twopi;
    if (th > theta[i] && th < hi) newth.push_back(th);
  }
  return newth;
}

template <class R>
void magnify_one(double s, double q, double rho_, double zre, double zim, double tol, int mode, const AdaptOpt& o,
                 double* out_mu, double* out_err, int32_t* out_n, uint32_t* out_status, double* out_theta /*optional, max_samples*/) {
  Contour<R> C;
  C.L = make_lens<R>(s, q);
  C.rho = (R)rho_;
  C.zc = Cx<R>((R)zre, (R)zim);
  C.twopi = R(2) * pi_v<R>();
  C.gate2 = R(o.slope_gate) * R(o.slope_gate);
  C.cos2 = R(o.slope_cos) * R(o.slope_cos);
  C.guard = o.hidden_guard;
  const R rtol = (R)tol;
  uint32_t status = 0;
  if (!(s > 0) || !(q > 0) || !(rho_ > 0) || !std::isfinite(s) || !std::isfinite(q) || !std::isfinite(rho_) ||
      !std::isfinite(zre) || !std::isfinite(zim)) {
    if (out_mu) *out_mu = std::numeric_limits<double>::quiet_NaN();
    if (out_err) *out_err = std::numeric_limits<double>::quiet_NaN();
    if (out_n) *out_n = 0;
    if (out_status) *out_status = 8;
    return;
  }
  if (s < 0.1 || s > 10 || q < 1e-9) status |= 8;   // outside the validated domain, P:374 (flagged, still computed)
  R A = 0, E = 0;
  int nbad = 0;
  if (mode == 0) {
    const int K = o.samples_per_iter;
    C.init(o.initial_samples);
    for (;;) {
      C.sums(A, E, nbad);
      const int n = (int)C.S.size();
      if (nbad == 0 && E <= rtol * std::abs(A)) { status |= 1; break; }           // P:272, A-1
      if (n + K > o.max_samples) { status |= 2; break; }                          // P:326, A-6
      // error-weighted inverse-transform sampling
      std::vector<R> th(n), er(n);
      std::vector<char> bad(n);
      for (int i = 0; i < n; ++i) { th[i] = C.S[i].theta; er[i] = C.P[i].err; bad[i] = (char)C.P[i].bad; }
      std::vector<R> newth = sampler_new_thetas(th, er, bad, C.twopi, rtol * std::abs(A), K, o.subtract_avg_tol);
      if (newth.empty()) { status |= 2; break; }
      C.insert(newth);
    }
  } else {
    C.init(256);
    for (;;) {
      C.sums(A, E, nbad);
      const int n = (int)C.S.size();
      if (nbad == 0 && E <= R(0.1) * rtol * std::abs(A)) { status |= 1; break; }
      if (n >= 65536) { status |= 2; break; }
      std::vector<int> idx(n);
      for (int i = 0; i < n; ++i) idx[i] = i;
      const int m = (n + 7) / 8;
      std::partial_sort(idx.begin(), idx.begin() + m, idx.end(), [&](int a, int b) {
        const R ea = C.P[a].bad ? std::numeric_limits<R>::infinity() : C.P[a].err;
        const R eb = C.P[b].bad ? std::numeric_limits<R>::infinity() : C.P[b].err;
        return ea > eb;
      });
      std::vector<R> newth;
      for (int k = 0; k < m; ++k) {
        const int i = idx[k];
        if (!C.P[i].bad && !(C.P[i].err > 0)) continue;
        newth.push_back(C.S[i].theta + R(0.5) * C.dtheta(i));
      }
      if (newth.empty()) { status |= 2; break; }
      C.insert(newth);
    }
  }
  int rep = 0, slp = 0, grd = 0;
  for (const auto& smp : C.S) {
    rep |= smp.repaired;
    slp |= smp.slope;
    grd |= smp.guard;
  }
  if (rep || nbad) status |= 4;
  if (grd) status |= 16;
  if (slp) status |= 32;
  if (out_mu) *out_mu = (double)(A / (pi_v<R>() * C.rho * C.rho));
  if (out_err) *out_err = (double)(E / std::abs(A));
  if (out_n) *out_n = (int32_t)C.S.size();
  if (out_status) *out_status = status;
  if (out_theta)
    for (size_t i = 0; i < C.S.size() && (int)i < o.max_samples; ++i) out_theta[i] = (double)C.S[i].theta;
}

// ---------------------------------------------------------------------------------------------------------
// N1: point-source adequacy tests, P:122 ("the quadrupole test and ghost image test check if the
// point-source approximation is accurate enough").  The paper prints no formulas; readings N1-a..c derive
// them from the lens equation:
//   N1-a  uniform disk: mu_fs = mu + (rho^2/8) Lap(mu) + O(rho^4), Lap = 4 d2/(dzeta dzetabar).  For one image, with
//         g, h, k the first three derivatives of f at the image and J = 1 - |g|^2: any F(z, zbar) has
//         dF/dzeta = (F_z - g F_zb)/J and dF/dzetabar = (F_zb - gbar F_z)/J (from dz/dzeta = 1/J, dz/dzetabar = -gbar/J).
//         Applied twice to F = 1/J.
//   N1-b  quadrupole test: sum_real rho^2/2 (|d2(1/J)/(dzeta dzetabar)| + |d2(1/J)/dzeta^2|) < c_Q * tol * A,  c_Q = 3.
//         The second, traceless derivative does not enter the disk average, but next to a cusp the Laplacian of a
//         bright image changes sign while the traceless part stays large: bounding both keeps the next order small.
//   N1-c  ghost-image test: a ghost root responds to a source shift delta by (delta - f'(w) conj(delta)) / (1 - f'(w) f'(z)),
//         w = conj(zeta) - f(z) (differentiate the 2-cycle); the pair becomes real when it closes its separation |R|:
//         rho (1 + |f'(w)|) / |1 - f'(w) f'(z)| < c_G |R|,  c_G = 0.1
// ---------------------------------------------------------------------------------------------------------
template <class R>
struct PsOut { int accept; R mu, qrel, A; int nreal; };

template <class R>
PsOut<R> point_source_test(double s, double q, double rho_, double zre, double zim, double tol) {
  const Lens<R> L = make_lens<R>(s, q);
  const R rho = (R)rho_;
  Sample<R> S;
  // the point source at the centre: theta is irrelevant for the images; rho = 0 puts the sample on the centre
  point_solve(L, Cx<R>((R)zre, (R)zim), R(0), R(0), S);
  const Cx<R> zeta((R)zre, (R)zim);
  const R z1 = L.z1, z2 = L.z2;                  // CM frame lens positions, Eq.(2)
  PsOut<R> o;
  o.accept = 1;
  o.nreal = S.nreal;
  R A = 0, Q = 0, Qabs = 0;
  for (int k = 0; k < 5; ++k) {
    const Cx<R> z = S.z[k];
    const Cx<R> a = R(1) / (z1 - z), b = R(1) / (z2 - z);
    const Cx<R> f = L.m1 * a + L.m2 * b;
    const Cx<R> g = L.m1 * a * a + L.m2 * b * b;
    if (S.kind[k] == 0) {   // N1-c
      const Cx<R> w = std::conj(zeta) - f;
      const Cx<R> aw = R(1) / (z1 - w), bw = R(1) / (z2 - w);
      const Cx<R> gw = L.m1 * aw * aw + L.m2 * bw * bw;
      const R resp = (R(1) + std::abs(gw)) / std::abs(Cx<R>(1, 0) - gw * g);
      if (!(rho * resp < R(0.1) * std::abs(S.Res[k]))) o.accept = 0;
      continue;
    }
    const Cx<R> h = R(2) * (L.m1 * a * a * a + L.m2 * b * b * b);
    const Cx<R> kk = R(6) * (L.m1 * a * a * a * a + L.m2 * b * b * b * b);
    const R J = R(1) - std::norm(g);
    // F = 1/J:  F_z = -J_z / J^2,  J_z = -h conj(g),  J_zb = -g conj(h)
    // first derivative  M = dF/dzeta = N / J^3,  N = h conj(g) - g^2 conj(h)
    const Cx<R> N = h * std::conj(g) - g * g * std::conj(h);
    const Cx<R> Nz = kk * std::conj(g) - R(2) * g * h * std::conj(h);
    const Cx<R> Nzb = h * std::conj(h) - g * g * std::conj(kk);
    const Cx<R> Jz = -h * std::conj(g), Jzb = -g * std::conj(h);
    const R J3 = J * J * J, J4 = J3 * J;
    const Cx<R> Mz = Nz / J3 - R(3) * N * Jz / J4;
    const Cx<R> Mzb = Nzb / J3 - R(3) * N * Jzb / J4;
    const Cx<R> d2 = (Mzb - std::conj(g) * Mz) / J;           // d2(1/J) / (dzeta dzetabar)
    const R p = (J > 0) ? R(1) : R(-1);
    A += p / J;
    Q += p * R(0.5) * rho * rho * d2.real();
    const Cx<R> t2 = (Mz - g * Mzb) / J;                       // d2(1/J) / dzeta^2, the traceless part
    Qabs += R(0.5) * rho * rho * (std::abs(d2) + std::abs(t2));
  }
  if (S.repaired) o.accept = 0;                                 // leave noise-floor cases to the contour
  o.A = A;
  o.mu = A + Q;
  o.qrel = Qabs / std::abs(A);
  if (!(Qabs < R(3) * (R)tol * std::abs(A))) o.accept = 0;      // N1-b
  if (!std::isfinite((double)o.mu) || !std::isfinite((double)o.qrel)) o.accept = 0;
  return o;
}

template <class R>
void point_out(double s, double q, double rho, double zre, double zim, double theta, double* z, double* Res,
                      double* J, int32_t* kind, double* zp, double* w, int32_t* info) {
  Lens<R> L = make_lens<R>(s, q);
  Sample<R> S;
  point_solve(L, Cx<R>((R)zre, (R)zim), (R)rho, (R)theta, S);
  for (int k = 0; k < 5; ++k) {
    z[2 * k] = (double)S.z[k].real();  z[2 * k + 1] = (double)S.z[k].imag();
    Res[2 * k] = (double)S.Res[k].real();  Res[2 * k + 1] = (double)S.Res[k].imag();
    J[k] = (double)S.J[k];
    kind[k] = S.kind[k];
    zp[2 * k] = (double)S.zp[k].real();  zp[2 * k + 1] = (double)S.zp[k].imag();
    w[k] = (double)S.w[k];
  }
  info[0] = S.nreal;
  info[1] = S.repaired;
  info[2] = S.sweeps;
}

}  // namespace

// =========================================================================================================
// C interface (ctypes).  All arrays are host arrays of double / int; complex = 2 consecutive doubles (re, im).
// =========================================================================================================
extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// Eq.(6) (form=6) or Eq.(4) (form=4) coefficients for source position zeta (CM frame).  out_c: 6 complex.
void orc_coeffs(double s, double q, double zre, double zim, int form, int prec, double* out_c) {
  if (prec) {
    typedef long double R;
    Lens<R> L = make_lens<R>(s, q);
    Cx<R> c[6];
    Cx<R> y = Cx<R>(zre, zim) - L.z2;
    if (form == 6) coeffs_eq6(y, L.s, L.m2, c); else coeffs_eq4(y, L.s, L.m1, L.m2, c);
    for (int i = 0; i < 6; ++i) { out_c[2 * i] = (double)c[i].real(); out_c[2 * i + 1] = (double)c[i].imag(); }
  } else {
    typedef double R;
    Lens<R> L = make_lens<R>(s, q);
    Cx<R> c[6];
    Cx<R> y = Cx<R>(zre, zim) - L.z2;
    if (form == 6) coeffs_eq6(y, L.s, L.m2, c); else coeffs_eq4(y, L.s, L.m1, L.m2, c);
    for (int i = 0; i < 6; ++i) { out_c[2 * i] = c[i].real(); out_c[2 * i + 1] = c[i].imag(); }
  }
}

// Roots of an arbitrary complex quintic (coefficients c0..c5) by the oracle's solver.
void orc_quintic_roots(const double* c_in, int prec, double* out_roots) {
  if (prec) {
    typedef long double R;
    Cx<R> c[6], r[5];
    for (int i = 0; i < 6; ++i) c[i] = Cx<R>(c_in[2 * i], c_in[2 * i + 1]);
    quintic_roots_dk(c, r);
    for (int k = 0; k < 5; ++k) { out_roots[2 * k] = (double)r[k].real(); out_roots[2 * k + 1] = (double)r[k].imag(); }
  } else {
    typedef double R;
    Cx<R> c[6], r[5];
    for (int i = 0; i < 6; ++i) c[i] = Cx<R>(c_in[2 * i], c_in[2 * i + 1]);
    quintic_roots_dk(c, r);
    for (int k = 0; k < 5; ++k) { out_roots[2 * k] = r[k].real(); out_roots[2 * k + 1] = r[k].imag(); }
  }
}

// One boundary point source: centre (zre, zim), radius rho, angle theta.
void orc_point(double s, double q, double rho, double zre, double zim, double theta, int prec, double* z, double* Res,
               double* J, int32_t* kind, double* zp, double* w, int32_t* info) {
  if (prec) point_out<long double>(s, q, rho, zre, zim, theta, z, Res, J, kind, zp, w, info);
  else point_out<double>(s, q, rho, zre, zim, theta, z, Res, J, kind, zp, w, info);
}

// Fixed-sampling face for a batch.  model_id may be NULL (then n_models is 1 or n_sources).
// out_z [n][N][5][2], out_kind [n][N][5], out_count [n][N], out_mu [n], out_err [n], out_ncross [n],
// out_piece [n][N][2] (dA, err per interval) -- every output pointer may be NULL.
void orc_images_fixed(int64_t n_models, const double* s, const double* q, const double* rho, int64_t n_sources,
                      const int32_t* model_id, const double* zeta, int N, int prec, int nthreads, double* out_z,
                      int8_t* out_kind, int8_t* out_count, double* out_mu, double* out_err, int32_t* out_ncross,
                      double* out_piece) {
  (void)nthreads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : orc_num_threads())
  for (int64_t i = 0; i < n_sources; ++i) {
    const int64_t m = model_id ? model_id[i] : (n_models == 1 ? 0 : i);
    double* oz = out_z ? out_z + size_t(i) * N * 10 : nullptr;
    int8_t* ok = out_kind ? out_kind + size_t(i) * N * 5 : nullptr;
    int8_t* oc = out_count ? out_count + size_t(i) * N : nullptr;
    double* op = out_piece ? out_piece + size_t(i) * N * 2 : nullptr;
    if (prec)
      images_fixed_one<long double>(s[m], q[m], rho[m], zeta[2 * i], zeta[2 * i + 1], N, oz, ok, oc, out_mu ? out_mu + i : nullptr,
                                    out_err ? out_err + i : nullptr, out_ncross ? out_ncross + i : nullptr, op);
    else
      images_fixed_one<double>(s[m], q[m], rho[m], zeta[2 * i], zeta[2 * i + 1], N, oz, ok, oc, out_mu ? out_mu + i : nullptr,
                               out_err ? out_err + i : nullptr, out_ncross ? out_ncross + i : nullptr, op);
  }
}

// Adaptive face for a batch.  mode 0 = the paper's sampler, mode 1 = the oracle's converged reference.
void orc_magnify(int64_t n_models, const double* s, const double* q, const double* rho, int64_t n_sources,
                 const int32_t* model_id, const double* zeta, double rel_tol, int mode, int samples_per_iter,
                 int initial_samples, int max_samples, int subtract_avg_tol, int prec, int nthreads, double* out_mu,
                 double* out_err, int32_t* out_nsamples, uint32_t* out_status, double slope_gate, double slope_cos,
                 int hidden_guard) {
  AdaptOpt o{samples_per_iter, initial_samples, max_samples, subtract_avg_tol, slope_gate, slope_cos, hidden_guard};
  (void)nthreads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads > 0 ? nthreads : orc_num_threads())
  for (int64_t i = 0; i < n_sources; ++i) {
    const int64_t m = model_id ? model_id[i] : (n_models == 1 ? 0 : i);
    if (prec)
      magnify_one<long double>(s[m], q[m], rho[m], zeta[2 * i], zeta[2 * i + 1], rel_tol, mode, o, out_mu ? out_mu + i : nullptr,
                               out_err ? out_err + i : nullptr, out_nsamples ? out_nsamples + i : nullptr,
                               out_status ? out_status + i : nullptr, nullptr);
    else
      magnify_one<double>(s[m], q[m], rho[m], zeta[2 * i], zeta[2 * i + 1], rel_tol, mode, o, out_mu ? out_mu + i : nullptr,
                          out_err ? out_err + i : nullptr, out_nsamples ? out_nsamples + i : nullptr,
                          out_status ? out_status + i : nullptr, nullptr);
  }
}

// N1: point-source adequacy tests over a batch.  out_accept[i] in {0,1}; out_mu = point source + quadrupole term;
// out_qrel = relative size of the quadrupole term; out_A = point-source magnification (sum of 1/|J| over real images).
void orc_point_source(int64_t n_models, const double* s, const double* q, const double* rho, int64_t n_sources,
                      const int32_t* model_id, const double* zeta, double rel_tol, int prec, int8_t* out_accept,
                      double* out_mu, double* out_qrel, double* out_A) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < n_sources; ++i) {
    const int64_t m = model_id ? model_id[i] : (n_models == 1 ? 0 : i);
    int acc;
    double mu, qr, A;
    if (prec) {
      const auto o = point_source_test<long double>(s[m], q[m], rho[m], zeta[2 * i], zeta[2 * i + 1], rel_tol);
      acc = o.accept; mu = (double)o.mu; qr = (double)o.qrel; A = (double)o.A;
    } else {
      const auto o = point_source_test<double>(s[m], q[m], rho[m], zeta[2 * i], zeta[2 * i + 1], rel_tol);
      acc = o.accept; mu = o.mu; qr = o.qrel; A = o.A;
    }
    if (out_accept) out_accept[i] = (int8_t)acc;
    if (out_mu) out_mu[i] = mu;
    if (out_qrel) out_qrel[i] = qr;
    if (out_A) out_A[i] = A;
  }
}

// Sorted sample angles the paper-style sampler ends with, for one source (diagnostics).  Returns n.
int orc_magnify_thetas(double s, double q, double rho, double zre, double zim, double rel_tol, int samples_per_iter,
                       int initial_samples, int max_samples, int subtract_avg_tol, int prec, double* out_theta) {
  AdaptOpt o{samples_per_iter, initial_samples, max_samples, subtract_avg_tol, 1e-5, 0.70710678118654752, 0};
  int32_t n = 0;
  if (prec) magnify_one<long double>(s, q, rho, zre, zim, rel_tol, 0, o, nullptr, nullptr, &n, nullptr, out_theta);
  else magnify_one<double>(s, q, rho, zre, zim, rel_tol, 0, o, nullptr, nullptr, &n, nullptr, out_theta);
  return n;
}

// ---- diagnostics for the pins (tests/test_oracle_errors.py); no arithmetic of their own --------------------------------

// The contour over an arbitrary sorted list of n boundary angles theta[] (0 <= theta_0 < ... < 2 pi): per interval
// (theta_i, theta_{i+1}) (the last one closes the loop) out_piece[i] = {dA, err}, out_terms[i][8] = Piece::terms,
// out_cross[i] = 0 / +1 creation / -1 annihilation; out_count[i] = real images of sample i.  Any output may be NULL.
void orc_pieces_at(double s, double q, double rho, double zre, double zim, int n, const double* theta, int prec,
                   double* out_piece, double* out_terms, int32_t* out_cross, int32_t* out_count) {
  auto run = [&](auto tag) {
    typedef decltype(tag) R;
    const Lens<R> L = make_lens<R>(s, q);
    std::vector<Sample<R>> S(n);
    for (int j = 0; j < n; ++j) point_solve(L, Cx<R>((R)zre, (R)zim), (R)rho, (R)theta[j], S[j]);
    const R twopi = R(2) * pi_v<R>();
    for (int j = 0; j < n; ++j) {
      const R dth = (j + 1 < n) ? (R)theta[j + 1] - (R)theta[j] : twopi - (R)theta[j] + (R)theta[0];
      Piece<R> P;
      eval_interval(S[j], S[(j + 1) % n], dth, P);
      if (out_piece) { out_piece[2 * j] = (double)P.dA; out_piece[2 * j + 1] = (double)P.err; }
      if (out_terms) for (int k = 0; k < 8; ++k) out_terms[8 * j + k] = (double)P.terms[k];
      if (out_cross) out_cross[j] = P.bad ? 99 : P.crossing;
      if (out_count) out_count[j] = S[j].nreal;
    }
  };
  if (prec) run((long double)0); else run((double)0);
}

// One interval between two SYNTHETIC samples given by the caller (kinds 0 / +1 / -1, positions z, derivatives z',
// z'^z'' per root; complex = (re, im)): what eval_interval makes of them.  out[0] = dA, out[1] = err, out[2..9] =
// Piece::terms; returns the crossing code (0, +1, -1; 99 = inconsistent).
int orc_eval_interval_synth(const int32_t* kindA, const double* zA, const double* zpA, const double* wA, const int32_t* kindB,
                            const double* zB, const double* zpB, const double* wB, double dth, double* out) {
  typedef long double R;
  Sample<R> A, B;
  for (int k = 0; k < 5; ++k) {
    A.kind[k] = kindA[k]; A.z[k] = Cx<R>(zA[2 * k], zA[2 * k + 1]); A.zp[k] = Cx<R>(zpA[2 * k], zpA[2 * k + 1]); A.w[k] = wA[k];
    B.kind[k] = kindB[k]; B.z[k] = Cx<R>(zB[2 * k], zB[2 * k + 1]); B.zp[k] = Cx<R>(zpB[2 * k], zpB[2 * k + 1]); B.w[k] = wB[k];
  }
  A.nreal = B.nreal = 0;
  for (int k = 0; k < 5; ++k) { A.nreal += A.kind[k] != 0; B.nreal += B.kind[k] != 0; }
  Piece<R> P;
  eval_interval(A, B, (R)dth, P);
  out[0] = (double)P.dA;
  out[1] = (double)P.err;
  for (int k = 0; k < 8; ++k) out[2 + k] = (double)P.terms[k];
  return P.bad ? 99 : P.crossing;
}

// One step of the paper's sampler on caller-given interval errors (sampler_new_thetas).  Returns the number of new
// angles written to out_theta (at most K).
int orc_sampler_step(int n, const double* theta, const double* err, double tolA, int K, int subtract_avg_tol, double* out_theta) {
  std::vector<double> th(theta, theta + n), er(err, err + n);
  std::vector<char> bad(n, 0);
  const std::vector<double> nt = sampler_new_thetas<double>(th, er, bad, 2.0 * pi_v<double>(), tolA, K, subtract_avg_tol);
  for (size_t i = 0; i < nt.size(); ++i) out_theta[i] = nt[i];
  return (int)nt.size();
}

// O9. Brute-force inverse ray shooting: rays on a uniform grid of nx x ny cells over the image-plane
// box [x0,x1] x [y0,y1]; a coarse cell is subdivided sub x sub when any of its corners or its centre lands
// within (rho + margin) of the source centre.  Returns the magnification (hit area / (pi rho^2)).
double orc_rayshoot(double s, double q, double rho, double zre, double zim, double x0, double x1, double y0, double y1,
                    int nx, int ny, int sub, int nthreads) {
  const Lens<double> L = make_lens<double>(s, q);
  const double hx = (x1 - x0) / nx, hy = (y1 - y0) / ny;
  auto map = [&](double x, double y, double& sx, double& sy) {
    // Eq.(1): zeta = z + m1/(conj z1 - conj z) + m2/(conj z2 - conj z)
    const double ax = x - L.z1, bx = x - L.z2;
    const double da = ax * ax + y * y, db = bx * bx + y * y;
    sx = x - L.m1 * ax / da - L.m2 * bx / db;
    sy = y - L.m1 * y / da - L.m2 * y / db;
  };
  double total = 0;
  (void)nthreads;
#pragma omp parallel for schedule(dynamic, 8) reduction(+ : total) num_threads(nthreads > 0 ? nthreads : orc_num_threads())
  for (int iy = 0; iy < ny; ++iy) {
    double rowsum = 0;
    for (int ix = 0; ix < nx; ++ix) {
      const double cx = x0 + ix * hx, cy = y0 + iy * hy;
      // distance of the mapped corners/centre from the source centre, and the local stretch of the map
      double dmin = 1e300, dmax = 0;
      double px[5] = {cx, cx + hx, cx, cx + hx, cx + 0.5 * hx}, py[5] = {cy, cy, cy + hy, cy + hy, cy + 0.5 * hy};
      double sxs[5], sys[5];
      for (int k = 0; k < 5; ++k) {
        map(px[k], py[k], sxs[k], sys[k]);
        const double d = std::hypot(sxs[k] - zre, sys[k] - zim);
        dmin = std::min(dmin, d);
        dmax = std::max(dmax, d);
      }
      double span = 0;
      for (int k = 0; k < 4; ++k) span = std::max(span, std::hypot(sxs[k] - sxs[4], sys[k] - sys[4]));
      if (!(dmin < rho + 2 * span) ) continue;           // whole cell maps outside the disk (with margin)
      if (std::isfinite(dmax) && dmax < rho - 2 * span && span < 0.25 * rho) { rowsum += hx * hy; continue; }   // wholly inside
      int hits = 0;
      for (int jy = 0; jy < sub; ++jy)
        for (int jx = 0; jx < sub; ++jx) {
          double sx, sy;
          map(cx + (jx + 0.5) * hx / sub, cy + (jy + 0.5) * hy / sub, sx, sy);
          const double ddx = sx - zre, ddy = sy - zim;
          hits += (ddx * ddx + ddy * ddy <= rho * rho);
        }
      rowsum += hx * hy * hits / double(sub * sub);
    }
    total += rowsum;
  }
  return total / (kPi * rho * rho);
}

}  // extern "C"
