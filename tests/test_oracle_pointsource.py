"""Pins of the point-source adequacy tests (readings N1-a..c in DESIGN.md) on the oracle side."""
import numpy as np
import pytest

import workloads as W
from oracle import api


def _one(s, q, rho, zc, tol=1e-4, prec=0):
    wl = W.Workload("t", np.array([s]), np.array([q]), np.array([rho]), np.zeros(1, np.int32),
                    np.array([[complex(zc).real, complex(zc).imag]]), tol)
    r = api.point_source(wl, tol, prec)
    return {k: v[0] for k, v in r.items()}, wl


@pytest.mark.parametrize("s,q,zc", [(1.3, 0.02, 0.31 + 0.17j), (0.8, 0.3, -0.4 + 0.55j), (2.2, 1e-3, 1.2 - 0.3j),
                                     (1.0, 0.1, 0.05 + 0.02j)])
def test_quadrupole_term_is_rho2_over_8_times_the_laplacian(s, q, zc):
    """N1-a: mu - A = (rho^2 / 8) Laplacian(A); the Laplacian is re-derived here by central differences of the
    oracle's own point-source magnification (inside a caustic too: the last case has five images)."""
    rho = 0.01
    h = 2e-4
    A = lambda z: _one(s, q, rho, z, prec=1)[0]["A"]
    lap = (A(zc + h) + A(zc - h) + A(zc + 1j * h) + A(zc - 1j * h) - 4.0 * A(zc)) / h ** 2
    r = _one(s, q, rho, zc, prec=1)[0]
    assert abs((r["mu"] - r["A"]) / (rho ** 2 / 8.0 * lap) - 1.0) < 1e-4


def test_quadrupole_single_lens_limit():
    """q -> 0: A(u) = (u^2+2)/(u sqrt(u^2+4)) (Paczynski); for a radial function Laplacian = A'' + A'/u, differentiated
    here in closed form."""
    u = 0.37
    rho = 0.02
    s, q = 1.7, 1e-9
    z1 = -q * s / (1 + q)
    r = _one(s, q, rho, z1 + u * np.exp(0.4j), prec=1)[0]
    A = (u * u + 2) / (u * np.sqrt(u * u + 4))
    A1 = -8.0 / (u * u * (u * u + 4) ** 1.5)
    A2 = 8.0 * (5 * u * u + 8) / (u ** 3 * (u * u + 4) ** 2.5)
    assert abs(r["A"] / A - 1) < 1e-6
    assert abs((r["mu"] - r["A"]) / (rho ** 2 / 8.0 * (A2 + A1 / u)) - 1) < 1e-4
    # and the uniform-disk value itself (independent: the oracle's converged contour) agrees to O(rho^4)
    ref = api.magnify(_one(s, q, rho, z1 + u * np.exp(0.4j))[1], 1e-8, mode=1)["mu"][0]
    assert abs(r["mu"] / ref - 1) < 5e-6 and abs(r["A"] / ref - 1) > 1e-4


def _sample(wl, k, seed):
    idx = np.sort(np.random.default_rng(seed).choice(wl.n_sources, min(k, wl.n_sources), replace=False))
    return wl.subset(idx)


@pytest.mark.parametrize("name,kw,k", [("config3", {}, 2500), ("config4", {}, 1500), ("config5", {}, 1500),
                                       ("fig5_map", dict(case="resonant"), 800), ("fig5_map", dict(case="wide"), 800),
                                       ("fig7_grid", {}, 1500), ("lowq_sweep", {}, 1000), ("config2", {}, 1000)])
def test_accepted_sources_are_within_tolerance(name, kw, k):
    """N1-b/c: every source the two tests accept is within the requested tolerance of the converged contour value
    -- in particular a source whose disk touches a caustic is never accepted (it would be off by far more)."""
    wl = _sample(W.get(name, **kw), k, 21)
    ref = api.magnify(wl, 1e-7, mode=1)["mu"]
    for tol in (1e-4, 1e-6):
        r = api.point_source(wl, tol)
        acc = r["accept"]
        err = np.abs(r["mu"] / ref - 1)
        assert np.all(err[acc] <= tol), (name, tol, err[acc].max())
    if name == "config3":
        assert api.point_source(wl, 1e-4)["accept"].mean() > 0.9      # most epochs are far from caustics
    if name == "lowq_sweep":
        assert api.point_source(wl, 1e-4)["accept"].mean() < 0.2      # placed on the planetary caustic


def test_point_source_double_and_long_double_agree():
    wl = _sample(W.config3(), 800, 5)
    a, b = api.point_source(wl, 1e-4, prec=0), api.point_source(wl, 1e-4, prec=1)
    assert (a["accept"] == b["accept"]).mean() > 0.995               # borderline cases may flip
    same = a["accept"] & b["accept"]
    assert np.abs(a["mu"][same] / b["mu"][same] - 1).max() < 1e-11
