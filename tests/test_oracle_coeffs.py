"""Pins of the oracle's coefficient builder and root finder (T-1, T-2).

The expected polynomial is obtained here, independently of Eq.(6), by eliminating conj(z) from the lens
equation Eq.(1) in the planet frame with 60-digit mpmath polynomial arithmetic.
"""
import mpmath as mp
import numpy as np
import pytest

from oracle import api

mp.mp.dps = 60


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


def elimination_poly(s, q, zeta):
    """Coefficients c0..c5 (mpc) of the quintic obtained by eliminating conj(eta) from
    y = eta - m1/(conj(eta)+s) - m2/conj(eta)  (Eq.(1) with planet at 0, primary at -s), normalised so that the
    leading coefficient is -conj(y)(conj(y)+s) like Eq.(6)."""
    s, q = mp.mpf(s), mp.mpf(q)
    m1, m2 = 1 / (1 + q), q / (1 + q)
    z2 = s / (1 + q)
    y = mp.mpc(zeta.real, zeta.imag) - z2
    yb = mp.conj(y)
    D = [mp.mpc(0), s, mp.mpc(1)]                      # eta (eta + s)
    # conj(eta) = N/D with N = conj(y) D + m1 eta + m2 (eta + s)
    N = _padd([yb * d for d in D], [m2 * s, m1 + m2])
    NsD = _padd(N, [s * d for d in D])
    G = _pmul(_pmul([-y, mp.mpc(1)], N), NsD)          # (eta - y) N (N + s D)
    G = _padd(G, [m1 * x for x in _pmul(N, D)], -1)    # - m1 N D
    G = _padd(G, [m2 * x for x in _pmul(NsD, D)], -1)  # - m2 (N + s D) D
    assert len(G) == 6
    return [-g for g in G]


def _rel(c, ref):
    return [float(abs(mp.mpc(complex(a).real, complex(a).imag) - b) / abs(b)) for a, b in zip(c, ref)]


CASES = [
    (1.0, 0.1, 0.2 + 0.2j),
    (0.5, 1e-6, -1.49981640625 - 0.0035j + 1e-4 * np.exp(2.6227j)),    # Fig.1 boundary point next to the cusp
    (0.5, 1e-6, -1.49981640625 + 0.0035j),
    (0.9, 1e-4, 0.01 + 0.003j),
    (3.0, 1e-4, 2.666 + 0.001j),
    (0.7, 1e-9, -0.728 + 0.0001j),
    (2.5, 0.5, -0.3 - 0.8j),
    (1.3, 3.0, 0.4 + 0.0j),                                            # Im zeta = 0 exactly, q > 1
]


@pytest.mark.parametrize("s,q,zeta", CASES)
def test_eq6_equals_elimination(s, q, zeta):
    """P-1: Eq.(6) as printed is the eliminated lens equation, coefficient by coefficient."""
    ref = elimination_poly(s, q, zeta)
    c_ld = api.coeffs(s, q, zeta, form=6, prec=1)      # long double, rounded to double on output
    c_d = api.coeffs(s, q, zeta, form=6, prec=0)
    assert max(_rel(c_ld, ref)) < 5e-16
    assert max(_rel(c_d, ref)) < 2e-13, _rel(c_d, ref)


def test_eq6_fp64_accuracy_low_q():
    """T-1 / P:116: near a planetary caustic at q = 1e-6 every Eq.(6) coefficient keeps ~14 digits in FP64."""
    rng = np.random.default_rng(7)
    worst = 0.0
    for _ in range(40):
        s = rng.uniform(0.4, 2.5)
        q = 10.0 ** rng.uniform(-7, -4)
        # planetary caustic sits near zeta = s - 1/s on the real axis (CM frame, up to O(q))
        zeta = (s - 1 / s) + np.sqrt(q) * (rng.uniform(-2, 2) + 1j * rng.uniform(-2, 2))
        ref = elimination_poly(s, q, zeta)
        worst = max(worst, max(_rel(api.coeffs(s, q, zeta, 6, 0), ref)))
    assert worst < 1e-12, worst


def test_eq4_foil_cancellation():
    """T-2 / P:92: the conventional form Eq.(4) (with the OCR repair E-1) is the same polynomial in exact
    arithmetic but loses digits ~ q^-1 in FP64, where Eq.(6) does not."""
    s, q = 0.5, 1e-6
    zeta = -1.49981640625 - 0.0035j + 1e-4 * np.exp(2.6227j)
    ref = elimination_poly(s, q, zeta)
    c4_ld = api.coeffs(s, q, zeta, form=4, prec=1)
    c4_d = api.coeffs(s, q, zeta, form=4, prec=0)
    c6_d = api.coeffs(s, q, zeta, form=6, prec=0)
    # same polynomial (long double Eq.(4) still shows its own cancellation, hence the loose bound)
    assert max(_rel(c4_ld, ref)) < 1e-10
    e4, e6 = _rel(c4_d, ref), _rel(c6_d, ref)
    assert e6[2] < 1e-13
    assert e4[2] > 1e-11 and e4[2] > 1e3 * e6[2], (e4, e6)   # >= 3 more digits lost in c2 than Eq.(6)


@pytest.mark.parametrize("prec", [0, 1])
def test_roots_backward_error_and_vieta(prec):
    """P-2: every root has a backward error at rounding level; Vieta's sum and product hold."""
    rng = np.random.default_rng(11)
    eps = 2.3e-16
    for trial in range(200):
        if trial < 100:
            c = rng.normal(size=6) + 1j * rng.normal(size=6)
        else:
            s = np.exp(rng.uniform(np.log(0.3), np.log(3)))
            q = np.exp(rng.uniform(np.log(1e-7), 0))
            c = api.coeffs(s, q, rng.uniform(-1.5, 1.5) + 1j * rng.uniform(-1.5, 1.5), 6, 1)
        r = api.quintic_roots(c, prec)
        for x in r:
            p = np.polyval(c[::-1], x)
            cond = np.polyval(np.abs(c[::-1]), abs(x))
            assert abs(p) <= 64 * eps * cond
        assert abs(r.sum() + c[4] / c[5]) <= 1e-12 * max(1.0, np.abs(r).max())
        assert abs(np.prod(r) + c[0] / c[5]) <= 1e-11 * max(abs(c[0] / c[5]), np.abs(r).max() ** 5 * 1e-3)


def test_roots_known_polynomial():
    """Roots of (x-1)(x-2)(x+3)(x-i)(x+2i) are recovered (textbook special case)."""
    roots = np.array([1, 2, -3, 1j, -2j])
    c = np.poly(roots)[::-1]
    r = api.quintic_roots(c, 0)
    for x in roots:
        assert np.abs(r - x).min() < 1e-13
