"""Pins of the oracle's crossing piece (Eq.(11)), error estimator (Eq.(17)-(18)), sampler and parity
repair (reading G-5) -- the parts round 1 left unpinned.  Every expected value comes from outside the oracle's
formulas: closed forms of a fold model, 60-digit mpmath image tracks obtained by eliminating conj(z) from Eq.(1),
fine integrations of the same interval, hand-computed quantiles of a toy weight vector, Eq.(7) itself.

Each test names the mutation of oracle/twk_oracle.cpp it is there to catch.
"""
import os

import mpmath as mp
import numpy as np
import pytest

import workloads as W
from oracle import api

GOLD = os.path.join(os.path.dirname(__file__), "golden")
T = {name: k for k, name in enumerate(api.TERMS)}


def paper_coefficients():
    """tests/golden/eq17_eq18_coefficients.txt: the numerical factors the paper prints in Eq.(10), (11), (17), (18)."""
    out = {}
    for line in open(os.path.join(GOLD, "eq17_eq18_coefficients.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, num, den = line.split()[:3]
        out[name] = float(num) / float(den)
    return out


# ---------------------------------------------------------------------------------------------------------------------
# (b) fold model: the image pair next to the critical curve, in closed form
# ---------------------------------------------------------------------------------------------------------------------
def _fold_samples(rng, creation, U, cubic=True):
    """Two synthetic samples around a fold crossing.  Next to the critical curve the two images of the pair are the
    points u = +sqrt(d) and u = -sqrt(d) of ONE smooth curve through the critical point (Schneider et al. 1992, cited
    P:255; Eq.(16) is its leading term), d = |theta - theta_c| being the distance of the sample from the crossing:
        z(u) = zc + a1 u + a2 u^2 + a3 u^3        (a1: across the critical curve, a2: along it; complex)
    so z' = z_u / (2u) dd/dtheta, z'' = (u z_uu - z_u) / (4 u^3), z'^z'' = z_u ^ z_uu / (8 u^3) dd/dtheta.
    Returns (A, B, dth, exact, par): `exact` = the exact contribution of the pair to the Stokes sum Eq.(8) -- the + track
    followed with increasing theta with weight +1, the - track with weight -1 (S-1), i.e. the line integral of
    1/2 z ^ dz from z- to z+ along the curve at a creation and from z+ to z- at an annihilation."""
    ang = rng.uniform(0, 2 * np.pi)
    a1 = rng.uniform(0.5, 2.0) * np.exp(1j * ang)
    a2 = rng.uniform(0.5, 2.0) * np.exp(1j * (ang + rng.choice([-1, 1]) * np.pi / 2 + rng.uniform(-0.5, 0.5)))
    a3 = (rng.uniform(0.5, 3.0) * np.exp(1j * rng.uniform(0, 2 * np.pi))) if cubic else 0.0
    zc = 0.3 * (rng.uniform(-1, 1) + 1j * rng.uniform(-1, 1))
    sg = +1.0 if creation else -1.0                       # dd / dtheta
    zpair, zp, w = [], [], []
    for u in (+U, -U):                                    # u > 0 is the positive-parity image
        zu = a1 + 2 * a2 * u + 3 * a3 * u * u
        zuu = 2 * a2 + 6 * a3 * u
        zpair.append(zc + a1 * u + a2 * u * u + a3 * u ** 3)
        zp.append(sg * zu / (2 * u))
        w.append(sg * (zu.real * zuu.imag - zu.imag * zuu.real) / (8 * u ** 3))
    still = [3 + 1j, -3 + 0.5j, 0.5 - 3j]                 # three ordinary images that do not move: zero-length links
    v = 0.3 + 0.1j
    three = dict(kind=[+1, -1, -1, 0, 0], z=still + [9 + 9j, 9 - 9j], zp=[v] * 5, w=[0.0] * 5)
    five = dict(kind=[+1, -1, -1, +1, -1], z=still + zpair, zp=[v] * 3 + zp, w=[0.0] * 3 + w)
    x, wt = np.polynomial.legendre.leggauss(8)            # exact for the polynomial integrand
    u = U * x
    z = zc + a1 * u + a2 * u ** 2 + a3 * u ** 3
    dz = a1 + 2 * a2 * u + 3 * a3 * u ** 2
    integral = 0.5 * np.sum(wt * (z.real * dz.imag - z.imag * dz.real)) * U      # u from -U (z-) to +U (z+)
    dth = U * U + rng.uniform(0.001, 0.05)
    par = dict(a1=a1, a2=a2, a3=a3, U=U)
    if creation:
        return three, five, dth, integral, par
    return five, three, dth, -integral, par


@pytest.mark.parametrize("creation", [True, False])
def test_fold_model_crossing_piece(creation):
    """Eq.(11) + reading S-2, and Eq.(18) + reading E-5, against the closed forms of the fold model.
    With d = U^2 -> 0:
      * tilde-Delta-theta -> 4 d and the printed correction -> (4/3) (a1 ^ a2) U^3 = the area between the pair's path and
        its chord: chord + correction reproduces the exact line integral up to a relative O(U^2) of the correction, at a
        creation AND at an annihilation, with Eq.(11) entering as printed in both;
      * E1 = c |w+ + w-| tdt^3 -> 96 c |a1 ^ a3| U^4          (c = 1/48: the sum, not the difference, of the two z'^z'')
      * E2 = c |(z+ - z-).(z'+ - z'-) -+ 2 |z+ - z-| sqrt|z'+ . z'-|| tdt -> 16 c |a2|^2 U^4   (c = 3/2; the leading
        terms 2 |a1|^2 cancel only with '-' at a creation and '+' at an annihilation)
      * E3 = c |dA^(p)| dtheta^2 (c = 1/10).
    Catches: correction sign at a creation / at an annihilation, chord direction, tilde-Delta-theta without the square
    root, any of the printed factors, E1 with the difference, the -+ rule swapped, a term dropped."""
    c = paper_coefficients()
    rng = np.random.default_rng(100 + creation)
    for U in (1e-2, 3e-3, 1e-3):
        for _ in range(10):
            A, B, dth, exact, p = _fold_samples(rng, creation, U)
            r = api.eval_interval_synth(A, B, dth)
            assert r["crossing"] == (1 if creation else -1)
            t = r["terms"]
            wedge12 = p["a1"].real * p["a2"].imag - p["a1"].imag * p["a2"].real
            wedge13 = p["a1"].real * p["a3"].imag - p["a1"].imag * p["a3"].real
            sliver = abs(t[T["corr"]])
            assert abs(sliver / (c["eq11"] * 32 * abs(wedge12) * U ** 3) - 1) < 100 * U * U + 1e-9
            assert abs(r["dA"] - exact) < 100 * U * U * sliver, (r["dA"], exact, sliver)
            assert abs(t[T["cE1"]] / (c["eq18_E1"] * 96 * abs(wedge13) * U ** 4) - 1) < 100 * U * U
            assert abs(t[T["cE2"]] / (c["eq18_E2"] * 16 * abs(p["a2"]) ** 2 * U ** 4) - 1) < 100 * U * U
            assert abs(t[T["cE3"]] / (c["eq18_E3"] * sliver * dth * dth) - 1) < 1e-12
            assert abs(r["err"] / (t[T["cE1"]] + t[T["cE2"]] + t[T["cE3"]]) - 1) < 1e-12       # reading A-2: the plain sum


def test_fold_model_estimate_bounds_the_error_of_the_piece():
    """What Eq.(18) is for: the piece's true error (chord + Eq.(11) against the exact line integral) is O(U^5), the
    estimate E1 + E2 is O(U^4): it bounds the true error over the whole range of sample distances the sampler meets."""
    rng = np.random.default_rng(3)
    for creation in (True, False):
        for U in (0.1, 0.03, 1e-2, 1e-3):
            for _ in range(10):
                A, B, dth, exact, p = _fold_samples(rng, creation, U)
                r = api.eval_interval_synth(A, B, dth)
                assert abs(r["dA"] - exact) < r["terms"][T["cE1"]] + r["terms"][T["cE2"]]


# ---------------------------------------------------------------------------------------------------------------------
# (c) crossing pieces of real lenses against a fine integration of the same interval
# ---------------------------------------------------------------------------------------------------------------------
CROSSING_GEOMETRIES = [
    (1.0, 0.1, 0.1, 0.2 + 0.2j),                    # Fig.2: two fold crossings of the resonant caustic
    (0.5, 1e-6, 1e-4, -1.49981640625 - 0.0035j),    # Fig.1: the boundary dips into a planetary-caustic cusp
    (1.6, 0.02, 0.03, 1.0 + 0.01j),                 # planetary caustic of a wide binary, straddled
    (0.5, 1e-4, 5e-5, -1.4992916666666667 + 0.03460833333333334j),   # Fig.5 left column: close-binary planetary caustic
    (0.8, 0.05, 0.06, -0.03 + 0.0j),                # central caustic of a close binary inside the disk
]


def _crossing_piece_errors(s, q, rho, zc, N, M=128):
    """Every crossing interval of the N-sample contour against the sum of the M pieces of its own subdivision
    (long double).  Returns rows (crossing code, |piece - fine| / |Eq.(11) correction|, |correction| / |A|)."""
    th = 2 * np.pi * np.arange(N) / N
    c = api.pieces_at(s, q, rho, zc, th, prec=1)
    A = c["dA"].sum()
    rows = []
    for i in np.nonzero(c["cross"])[0]:
        lo, hi = th[i], (th[i + 1] if i + 1 < N else 2 * np.pi)
        sub = lo + (hi - lo) * np.arange(M + 1) / M
        if i + 1 == N:
            continue                                     # keep the sub-grid sorted: skip the wrap-around interval
        # the fine contour over [lo, hi] only: evaluate the sub-grid plus the rest of the coarse grid, take its pieces
        grid = np.concatenate([th[: i + 1], sub[1:-1], th[i + 1:]])
        f = api.pieces_at(s, q, rho, zc, grid, prec=1)
        fine = f["dA"][i: i + M].sum()
        if np.abs(f["cross"][i: i + M]).sum() != 1:      # more than one crossing inside: not what the piece models
            continue
        corr = c["terms"][i, T["corr"]]
        rows.append((int(c["cross"][i]), abs(c["dA"][i] - fine) / abs(corr), abs(corr / A)))
    return rows


def test_crossing_pieces_against_fine_integration():
    """Eq.(11) + S-2 on real lenses: with the correction the crossing piece is closer to the fine integration of the same
    interval than the bare chord is, by a wide margin, at creations AND at annihilations (a flipped sign leaves the
    piece two corrections away).  Catches: correction sign at a creation / at an annihilation, each on its own."""
    stats = {+1: [], -1: []}
    for s, q, rho, zc in CROSSING_GEOMETRIES:
        for N in (160, 200, 256, 300):
            for code, rel, size in _crossing_piece_errors(s, q, rho, zc, N):
                if size > 1e-9:                          # the correction itself is above rounding
                    stats[code].append(rel)
    for code in (+1, -1):
        r = np.array(stats[code])
        assert len(r) >= 12, (code, len(r))
        assert np.median(r) < 0.2, (code, np.median(r))
        assert np.mean(r < 0.6) > 0.9, (code, np.sort(r)[-5:])


# ---------------------------------------------------------------------------------------------------------------------
# (a) Eq.(17) term by term against 60-digit image tracks (mpmath elimination of Eq.(1), independent of the oracle)
# ---------------------------------------------------------------------------------------------------------------------
mp.mp.dps = 50


def _pmul(a, b):
    out = [mp.mpc(0)] * (len(a) + len(b) - 1)
    for i, x in enumerate(a):
        for j, y in enumerate(b):
            out[i + j] += x * y
    return out


def _padd(a, b, sb=1):
    n = max(len(a), len(b))
    a = list(a) + [mp.mpc(0)] * (n - len(a))
    b = list(b) + [mp.mpc(0)] * (n - len(b))
    return [x + sb * y for x, y in zip(a, b)]


def _mp_images(s, q, zeta):
    """The real images of the point source zeta (CM frame) from Eq.(1) alone: eliminate conj(eta) in the planet frame
    (planet at 0, primary at -s), solve the quintic with mpmath, keep the roots that satisfy Eq.(1)."""
    s, q = mp.mpf(s), mp.mpf(q)
    m1, m2 = 1 / (1 + q), q / (1 + q)
    z2 = s / (1 + q)
    y = zeta - z2
    yb = mp.conj(y)
    D = [mp.mpc(0), s, mp.mpc(1)]
    N = _padd([yb * d for d in D], [m2 * s, m1 + m2])
    NsD = _padd(N, [s * d for d in D])
    G = _pmul(_pmul([-y, mp.mpc(1)], N), NsD)
    G = _padd(G, [m1 * x for x in _pmul(N, D)], -1)
    G = _padd(G, [m2 * x for x in _pmul(NsD, D)], -1)
    roots = mp.polyroots(G[::-1], maxsteps=200, extraprec=200)
    out = []
    for eta in roots:
        res = y - eta + m1 / mp.conj(eta + s) + m2 / mp.conj(eta)
        if abs(res) < mp.mpf(10) ** -30:
            out.append(eta + z2)
    return out


def _track_derivatives(s, q, rho, zc, theta, k=mp.mpf(1) / 400):
    """z, z', z'', z''', z'''' of every real image at boundary angle theta, by 9-point central differences of the mpmath
    image positions (positions only: no f', no J).  Returns a list of 5-tuples of Python complex."""
    pts = []
    for j in range(-4, 5):
        t = mp.mpf(theta) + j * k
        zeta = mp.mpc(zc.real, zc.imag) + mp.mpf(rho) * mp.expj(t)
        pts.append(_mp_images(s, q, zeta))
    assert all(len(p) == len(pts[4]) for p in pts)
    tracks = []
    for z0 in pts[4]:
        tr, cur = {0: z0}, z0
        for j in range(1, 5):
            cur = min(pts[4 + j], key=lambda z: abs(z - cur))
            tr[j] = cur
        cur = z0
        for j in range(1, 5):
            cur = min(pts[4 - j], key=lambda z: abs(z - cur))
            tr[-j] = cur
        f = [tr[j] for j in range(-4, 5)]
        # 9-point central stencils (standard finite-difference weights, accuracy order 8 / 8 / 6 / 6)
        c1 = [mp.mpf(x) for x in (1 / mp.mpf(280), -4 / mp.mpf(105), 1 / mp.mpf(5), -4 / mp.mpf(5), 0, 4 / mp.mpf(5), -1 / mp.mpf(5), 4 / mp.mpf(105), -1 / mp.mpf(280))]
        c2 = [mp.mpf(x) for x in (-1 / mp.mpf(560), 8 / mp.mpf(315), -1 / mp.mpf(5), 8 / mp.mpf(5), -205 / mp.mpf(72), 8 / mp.mpf(5), -1 / mp.mpf(5), 8 / mp.mpf(315), -1 / mp.mpf(560))]
        c3 = [mp.mpf(x) for x in (-7 / mp.mpf(240), 3 / mp.mpf(10), -169 / mp.mpf(120), 61 / mp.mpf(30), 0, -61 / mp.mpf(30), 169 / mp.mpf(120), -3 / mp.mpf(10), 7 / mp.mpf(240))]
        c4 = [mp.mpf(x) for x in (7 / mp.mpf(240), -2 / mp.mpf(5), 169 / mp.mpf(60), -122 / mp.mpf(15), 91 / mp.mpf(8), -122 / mp.mpf(15), 169 / mp.mpf(60), -2 / mp.mpf(5), 7 / mp.mpf(240))]
        d = [sum(c * x for c, x in zip(cc, f)) / k ** n for n, cc in ((1, c1), (2, c2), (3, c3), (4, c4))]
        tracks.append(tuple(complex(x) for x in [z0] + d))
    return tracks


def _wedge(a, b):
    return a.real * b.imag - a.imag * b.real


def _dot(a, b):
    return a.real * b.real + a.imag * b.imag


SMOOTH_ARCS = [(0.9, 0.2, 0.05, 0.6 + 0.4j, 1.1), (1.4, 0.03, 0.08, -0.5 + 0.3j, 4.0), (0.7, 0.5, 0.1, 0.1 - 0.9j, 2.5)]


@pytest.mark.parametrize("s,q,rho,zc,theta_m", SMOOTH_ARCS)
def test_eq17_terms_against_independent_tracks(s, q, rho, zc, theta_m):
    """Eq.(17) on a smooth arc.  With z_k the k-th theta-derivative of an image track at the interval's
    midpoint and h the interval, Taylor expansion of the printed expressions gives
        E1 -> c1 |z1 ^ z3| h^4,                       c1 = 1/48   (w' = z1 ^ z3)
        E2 -> c2 c10/2 |z1 ^ z2| | |z2|^2/4 - z1.z3/6 | / |z1|^2 h^5,   c2 = 3/2, c10 = 2 * (1/24) = 1/12 of dA^(p)
        E3 -> c3 c10 |z1 ^ z2| h^5 ... (c3 = 1/10; dA^(p) -> (1/12) z1 ^ z2 h^3)
        E4 -> |z1 ^ z4 + 2 z2 ^ z3| h^5 / 144        (dA^(p1) - dA^(p2), from the 1/24 and 1/12 of Eq.(10))
    summed over the interval's links.  The derivatives come from mpmath image tracks (elimination of Eq.(1), positions
    only); the factors from the paper's print (tests/golden).  Catches: E1 1/48 -> 1/96, E2 / E3 / E4 dropped or
    rescaled, a wrong z' or z'^z'' inside them."""
    c = paper_coefficients()
    h = 2 * np.pi / 1024
    r = api.pieces_at(s, q, rho, zc, [theta_m - h / 2, theta_m + h / 2], prec=1)
    tracks = _track_derivatives(s, q, rho, zc, theta_m)
    assert len(tracks) == 3 and r["count"][0] == 3
    dAp = c["eq10_p1"] * 2          # dA^(p) -> 2 * (1/24) (z1 ^ z2) h^3 on a smooth arc
    E1 = sum(c["eq17_E1"] * abs(_wedge(z1, z3)) * h ** 4 for _, z1, z2, z3, z4 in tracks)
    E2 = sum(c["eq17_E2"] * dAp * abs(_wedge(z1, z2)) * abs(abs(z2) ** 2 / 4 - _dot(z1, z3) / 6) / abs(z1) ** 2 * h ** 5
             for _, z1, z2, z3, z4 in tracks)
    E3 = sum(c["eq17_E3"] * dAp * abs(_wedge(z1, z2)) * h ** 5 for _, z1, z2, z3, z4 in tracks)
    E4 = sum(abs(_wedge(z1, z4) + 2 * _wedge(z2, z3)) * h ** 5 / 144 for _, z1, z2, z3, z4 in tracks)
    got = r["terms"][0]
    for name, want in (("E1", E1), ("E2", E2), ("E3", E3), ("E4", E4)):
        assert abs(got[T[name]] / want - 1) < 0.02, (name, got[T[name]], want)
    assert abs(r["err"][0] / (E1 + E2 + E3 + E4) - 1) < 0.02                      # reading A-2: the plain sum
    # and the area piece itself: beyond the trapezium (taken from the mpmath end points) the oracle adds dA^(p) =
    # (1/12) z1 ^ z2 h^3 + (h^5 / 480)(z1 ^ z4 - z2 ^ z3)   [= exact arc - trapezium]   + (h^5 / 1440)(7 z1^z4 + 8 z2^z3)
    par = _parities(s, q, tracks)
    ends = []
    for sg in (-1, +1):
        zeta = mp.mpc(zc.real, zc.imag) + mp.mpf(rho) * mp.expj(mp.mpf(theta_m) + sg * mp.mpf(h) / 2)
        imgs = [complex(z) for z in _mp_images(s, q, zeta)]
        ends.append([min(imgs, key=lambda z: abs(z - (z0 + sg * z1 * h / 2))) for z0, z1, _, _, _ in tracks])
    trap = sum(p * 0.5 * _wedge(a, b - a) for p, a, b in zip(par, ends[0], ends[1]))
    para = sum(p * (_wedge(z1, z2) * h ** 3 / 12 + (_wedge(z1, z4) - _wedge(z2, z3)) * h ** 5 / 480
                    + (7 * _wedge(z1, z4) + 8 * _wedge(z2, z3)) * h ** 5 / 1440) for p, (_, z1, z2, z3, z4) in zip(par, tracks))
    assert abs((r["dA"][0] - trap) / para - 1) < 1e-6, (r["dA"][0] - trap, para)


def _parities(s, q, tracks):
    m1, m2 = 1 / (1 + q), q / (1 + q)
    z1l, z2l = -q * s / (1 + q), s / (1 + q)
    return [np.sign(1 - abs(m1 / (z1l - t[0]) ** 2 + m2 / (z2l - t[0]) ** 2) ** 2) for t in tracks]


HONESTY_CASES = [(1.0, 0.1, 0.1, 0.2 + 0.2j), (1.0, 0.1, 0.01, 0.303 + 0.0j), (0.9, 1e-4, 1e-3, 0.004 + 0.0005j),
                 (3.0, 1e-4, 1e-4, 2.6664 + 0.0002j), (0.5, 1e-6, 1e-4, -1.49981640625 - 0.0035j),
                 (1.4113848311835726, 0.5319220188997608, 0.008902655845331566, -0.30393401 - 0.2187177j)]


def test_interval_estimates_are_honest_on_adaptive_grids():
    """P:272 / P:344: what the stop rule compares with the tolerance.  On the sample sets the paper-style sampler ends
    with at tol 1e-4, every interval is integrated again on its own 64-fold subdivision (long double): (i) an interval's
    estimate falls below its true error only marginally -- the whole shortfall, sum of max(true_i - e_i, 0), stays below
    the estimate total (so the true error of a converged source is < 2 tol) and below tol |A|; (ii) the estimate is not
    vacuous: sum e_i <= 60 sum true_i.  Catches: any of E1..E4 of Eq.(17) or E1..E2 of Eq.(18) dropped (the estimate of
    the intervals that term dominates falls below their true error), a gross over-estimate."""
    for s, q, rho, zc in HONESTY_CASES:
        th = api.magnify_thetas(s, q, rho, zc, 1e-4)
        n, M = len(th), 64
        c = api.pieces_at(s, q, rho, zc, th)
        ext = np.concatenate([th, [2 * np.pi]])
        fine = (ext[:-1, None] + (ext[1:] - ext[:-1])[:, None] * np.arange(M)[None, :] / M).ravel()
        f = api.pieces_at(s, q, rho, zc, fine, prec=1)
        true = np.abs(c["dA"] - f["dA"].reshape(n, M).sum(1))
        A = abs(f["dA"].sum())
        assert c["err"].sum() <= 1e-4 * abs(c["dA"].sum())
        short = np.maximum(true - c["err"], 0.0).sum()
        assert short < 1e-4 * A and short < c["err"].sum(), (s, q, rho, zc, short / A, c["err"].sum() / A)
        assert true.sum() < c["err"].sum(), (c["err"].sum() / A, true.sum() / A)


# ---------------------------------------------------------------------------------------------------------------------
# (d) sampler: quantile placement, average tolerance
# ---------------------------------------------------------------------------------------------------------------------
def test_sampler_toy_quantiles_by_hand():
    """P:304, Fig.4: inverse transform of the normalised cumulative error with linear interpolation.  Four
    intervals of a quarter turn with errors 1, 3, 0, 4 (total 8) and 8 quantiles, no tolerance subtraction: the quantile
    levels are (k + 1/2) of the total (reading A-4), so interval 0 (cumulative 0..1) receives 0.5 -> half way;
    interval 1 (1..4) receives 1.5, 2.5, 3.5 -> 1/6, 1/2, 5/6 of the way; interval 2 nothing; interval 3 (4..8) receives
    4.5 .. 7.5 -> 1/8, 3/8, 5/8, 7/8.  Worked out by hand from the paper's description, not from the code.
    Catches: quantiles at (k + 1)/K or k/K, interpolation against the wrong interval, a cumulative sum off by one."""
    q = np.pi / 2
    got = api.sampler_step([0, q, 2 * q, 3 * q], [1.0, 3.0, 0.0, 4.0], 0.0, K=8, subtract_avg_tol=0)
    want = np.array([0.5, 1 + 1 / 6, 1.5, 1 + 5 / 6, 3.125, 3.375, 3.625, 3.875]) * q
    assert len(got) == 8 and np.allclose(got, want, rtol=0, atol=1e-14)


def test_sampler_k_quantiles_give_k_new_samples():
    """Fig.4's caption: "The inverse transform method generates eight new samples" from eight quantiles.  With
    every weight positive, K quantiles uniform on the vertical axis must give K distinct NEW angles strictly inside
    intervals -- true for levels (k + 1/2)/K, false for k/K (the first lands on theta_0) and (k + 1)/K (the last lands
    on 2 pi = theta_0).  Catches: the quantile offset of reading A-4."""
    rng = np.random.default_rng(4)
    for K in (8, 64):
        th = np.sort(rng.uniform(0, 2 * np.pi, 40))
        th[0] = 0.0
        err = rng.uniform(0.1, 1.0, 40)
        new = api.sampler_step(th, err, 0.0, K=K, subtract_avg_tol=0)
        assert len(new) == K and len(np.unique(new)) == K
        assert np.all(np.diff(new) > 0) and new[0] > 0 and new[-1] < 2 * np.pi
        assert not np.isin(new, th).any()
        # uniform weights per unit angle -> the new angles are uniform in angle: (k + 1/2) 2 pi / K
        uni = api.sampler_step(th, np.diff(np.concatenate([th, [2 * np.pi]])), 0.0, K=K, subtract_avg_tol=0)
        assert np.allclose(uni, (np.arange(K) + 0.5) * 2 * np.pi / K, atol=1e-12)


def test_sampler_average_tolerance_by_hand():
    """"we subtract each error by the average tolerance ... if the error between (theta_i, theta_i+1) is
    already lower than expected, no more points needed to be added here" (reading A-5: average = tol |A| / n).
    Errors 1.2, 2.1, 0.45, 4.25 (total 8) with tol |A| = 2 over n = 4 intervals: average 0.5, weights 0.7, 1.6, 0, 3.75
    (total 6.05); 8 quantiles at (k + 1/2) 6.05 / 8.  Interval 2 (0.45 < 0.5) gets nothing; without the subtraction its
    cumulative range 3.3..3.75 holds the level 3.5 and it would.
    Catches: the subtraction switched off, subtracting tol |A| instead of its average, no clamp at zero."""
    q = np.pi / 2
    th = [0, q, 2 * q, 3 * q]
    e = [1.2, 2.1, 0.45, 4.25]
    got = api.sampler_step(th, e, 2.0, K=8, subtract_avg_tol=1)
    lev = (np.arange(8) + 0.5) * 6.05 / 8
    want = []
    for x in lev:
        if x < 0.7:
            want.append((x / 0.7) * q)
        elif x < 2.3:
            want.append(q + (x - 0.7) / 1.6 * q)
        else:
            want.append(3 * q + (x - 2.3) / 3.75 * q)
    assert np.allclose(got, want, rtol=0, atol=1e-14)
    assert not np.any((got > 2 * q) & (got < 3 * q))
    off = api.sampler_step(th, e, 2.0, K=8, subtract_avg_tol=0)
    assert np.any((off > 2 * q) & (off < 3 * q))


def test_sampler_beats_uniform_refinement():
    """P:304-312 as a whole, on the Fig.2 source: to bring the error estimate below 1e-5 (the stop rule)
    the error-weighted sampler needs several times fewer samples than uniform sampling, and its result is that accurate.
    (The average-tolerance trick is pinned by the toy above: with 64 samples per iteration its effect on the sample COUNT
    of real sources is below the granularity -- measured on 80 caustic-crossing sources: 17,280 samples with it, 17,088
    without.)  Catches: weights not following the error."""
    wl = W.fig2_case()
    truth = api.magnify(wl, 1e-8, mode=1, prec=1)["mu"][0]
    r = api.magnify(wl, 1e-5, mode=0)
    assert abs(r["mu"][0] / truth - 1) < 1e-5
    n_adapt = int(r["nsamples"][0])
    n_uni = next(N for N in (256, 512, 1024, 2048, 4096, 8192, 16384) if api.images_fixed(wl, N)["err"][0] <= 1e-5)
    assert n_uni >= 4 * n_adapt, (n_uni, n_adapt)


# ---------------------------------------------------------------------------------------------------------------------
# (e) parity repair (reading G-5)
# ---------------------------------------------------------------------------------------------------------------------
def _caustic_points(s, q, n_phi):
    """Points of the caustic: critical-curve points z with f'(z) = e^{-i phi} (|f'| = 1, Eq.(7)), i.e. the quartic
    m1 (z2 - z)^2 + m2 (z1 - z)^2 = e^{-i phi} (z1 - z)^2 (z2 - z)^2, mapped through Eq.(1)."""
    m1, m2 = 1 / (1 + q), q / (1 + q)
    z1, z2 = -q * s / (1 + q), s / (1 + q)
    out = []
    for phi in 2 * np.pi * (np.arange(n_phi) + 0.5) / n_phi:
        e = np.exp(-1j * phi)
        p1sq, p2sq = np.polymul([-1, z1], [-1, z1]), np.polymul([-1, z2], [-1, z2])
        poly = np.polysub(e * np.polymul(p1sq, p2sq), np.polyadd(m1 * p2sq, m2 * p1sq))
        for z in np.roots(poly):
            for _ in range(3):                                  # Newton polish on the quartic itself
                z = z - np.polyval(poly, z) / np.polyval(np.polyder(poly), z)
            out.append(z + np.conj(m1 / (z1 - z) + m2 / (z2 - z)))
    return np.array(out)


def test_parity_repair_flips_the_smallest_jacobian():
    """P:155 (parity sum -1) + Eq.(7) (p = sign J).  A point source ON the caustic (to double rounding) has an image pair
    on the critical curve whose J ~ +-1e-8 is below the rounding of its own position: when both come out with the same
    sign the parity sum is broken, and only re-signing one of THAT pair is consistent with Eq.(7) for every image whose
    |J| is well above rounding.  Catches: the repair flipping the largest |J| (or any well-conditioned image)."""
    fired = 0
    for s, q in ((1.0, 0.1), (0.8, 0.02), (1.5, 0.3), (1.0, 1.0)):
        for zeta in _caustic_points(s, q, 150):
            p = api.point(s, q, 0.0, zeta, 0.0, 0)
            real = p["kind"] != 0
            assert p["kind"][real].sum() == -1
            if not p["repaired"]:
                continue
            fired += 1
            solid = real & (np.abs(p["J"]) > 1e-4)
            assert np.all(p["kind"][solid] == np.sign(p["J"][solid])), (s, q, zeta, p["J"], p["kind"])
    assert fired >= 10, fired


# ---------------------------------------------------------------------------------------------------------------------
# B-1: a boundary sample exactly on a lens
# ---------------------------------------------------------------------------------------------------------------------
def test_boundary_sample_on_a_lens_is_continuous():
    """Reading B-1: with a boundary sample EXACTLY on a lens the quintic loses its leading coefficient (c5 = -conj(y) v_c
    = 0, Eq.(6)); the oracle moves such a sample off the lens by 1e-14 s.  The magnification is a continuous function of
    the source position there, so the result must agree with sources shifted by ~1e-9 in any direction (which never
    trigger the rule) to the accuracy asked for, and carry status bit 16."""
    cases = [(1.0, 1.0, 0.25, 0.25 + 0j), (1.0, 1.0, 0.25, 0.5 - 0.25j), (1.0, 1.0, 0.25, -0.25 + 0j),
             (0.8, 0.25, 0.125, -0.285 + 0j), (1.0, 0.5, 0.25, 1 / 1.5 - 0.25 + 0j)]
    for s, q, rho, zc in cases:
        z = np.array([zc, zc + 1e-9, zc - 1e-9j, zc + 3e-9 + 2e-9j])
        wl = W.Workload("b1", np.array([s]), np.array([q]), np.array([rho]), np.zeros(4, np.int32),
                        np.stack([z.real, z.imag], 1).copy(), 1e-6)
        for mode in (0, 1):
            r = api.magnify(wl, 1e-6, mode=mode)
            assert np.all(np.isfinite(r["mu"])) and np.all(r["status"] & 1)
            assert r["status"][0] & 16 and not np.any(r["status"][1:] & 16)
            assert np.abs(r["mu"][0] / r["mu"][1:] - 1).max() < 1e-6
        # the sample on the lens: two of the five roots are the degenerate ones (on the pole, run away), both ghosts
        hit = 0
        for th in (0.0, np.pi / 2, np.pi, 1.5 * np.pi):
            zj = zc + rho * complex(np.cos(th), np.sin(th))
            if min(abs(zj - s / (1 + q)), abs(zj + q * s / (1 + q))) < 1e-15:
                p = api.point(s, q, rho, zc, th, 0)
                assert p["nreal"] == 3 and np.abs(p["z"][p["kind"] == 0]).max() > 1e12
                hit += 1
        assert hit >= 1


# ---------------------------------------------------------------------------------------------------------------------
# L-4 guard (extension): hidden double crossings
# ---------------------------------------------------------------------------------------------------------------------
L4_SOURCES = [(0.5, 1e-4, 5e-5, -1.500225 + 0.03455833333333334j),       # Fig.5 close map, grazes a fold
              (1.0, 0.1, 0.01, -0.15087891 + 0.30615234j),               # BASELINE config 4 grid point and its mirror image
              (1.0, 0.1, 0.01, -0.15087891 - 0.30615234j)]


def test_hidden_crossing_guard():
    """Reading L-4.  These three sources dip into the caustic and out again between two of the first 64 samples: Eq.(17)
    cannot see it and the paper-style sampler stops at 64 samples, 2-6 tolerances off.  With the guard the hidden area
    (predicted from the ghost pair's separation at the neighbouring samples) enters the estimate, the sampler refines
    there and the result is within the tolerance of the converged reference.  On sources without a hidden crossing the
    guard changes nothing (same sample sets, bit-identical values)."""
    for s, q, rho, zc in L4_SOURCES:
        wl = W.Workload("l4", np.array([s]), np.array([q]), np.array([rho]), np.zeros(1, np.int32),
                        np.array([[zc.real, zc.imag]]), 1e-4)
        ref = api.magnify(wl, 1e-7, mode=1, prec=1, hidden_guard=1)["mu"][0]
        off = api.magnify(wl, 1e-4, mode=0)
        on = api.magnify(wl, 1e-4, mode=0, hidden_guard=1)
        assert off["nsamples"][0] == 64 and abs(off["mu"][0] / ref - 1) > 1.5e-4
        assert on["nsamples"][0] > 64 and abs(on["mu"][0] / ref - 1) < 1e-5
    wl = W.config3(n_models=300, n_epochs=20)
    a, b = api.magnify(wl, 1e-4, mode=0), api.magnify(wl, 1e-4, mode=0, hidden_guard=1)
    assert np.array_equal(a["nsamples"], b["nsamples"]) and np.array_equal(a["mu"], b["mu"])
    # fine sampling of the interval confirms what the guard predicted: two crossings inside one first-iteration interval
    s, q, rho, zc = L4_SOURCES[0]
    coarse = api.pieces_at(s, q, rho, zc, 2 * np.pi * np.arange(64) / 64)
    fine = api.pieces_at(s, q, rho, zc, 2 * np.pi * np.arange(64 * 64) / (64 * 64))
    assert np.all(coarse["count"] == 3) and np.abs(fine["cross"]).reshape(64, 64).sum(1).max() == 2
