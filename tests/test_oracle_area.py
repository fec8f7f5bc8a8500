"""Pins of the oracle's linker / integrator / error estimate / samplers against closed
forms, brute force and the paper's worked examples.  Expected values are computed here or are the paper's."""
import os

import numpy as np
import pytest

import workloads as W
from oracle import api

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _one(s, q, rho, zeta, tol=1e-6, fixed_n=0):
    z = np.array([[complex(zeta).real, complex(zeta).imag]])
    return W.Workload("t", np.array([float(s)]), np.array([float(q)]), np.array([float(rho)]), np.zeros(1, np.int32), z, tol,
                      fixed_n)


def mu_ref(s, q, rho, zeta, tol=1e-7, prec=1):
    return api.magnify(_one(s, q, rho, zeta), tol, mode=1, prec=prec)["mu"][0]


def single_lens_disk_mu(u, rho, n=200001):
    """Uniform disk behind ONE point lens of unit mass: area enclosed by the exact image boundaries
    z+- = zeta/2 (1 +- sqrt(1 + 4/|zeta|^2)) (textbook), by the periodic trapezoid rule (spectrally accurate)."""
    th = 2 * np.pi * np.arange(n) / n
    zeta = u + rho * np.exp(1j * th)
    dzeta = 1j * rho * np.exp(1j * th)
    r2 = np.abs(zeta) ** 2
    root = np.sqrt(1 + 4 / r2)
    droot = (-4 / r2**2) * (zeta.real * dzeta.real + zeta.imag * dzeta.imag) / root      # d/dtheta sqrt(1+4/|zeta|^2)
    area = 0.0
    for sg in (+1, -1):
        z = 0.5 * zeta * (1 + sg * root)
        dz = 0.5 * dzeta * (1 + sg * root) + 0.5 * zeta * sg * droot
        area += sg * 0.5 * np.sum(z.real * dz.imag - z.imag * dz.real) * (2 * np.pi / n)
    return area / (np.pi * rho**2)


def test_single_lens_quadrature_helper_matches_closed_form_at_u0():
    """Sanity of the helper itself: u = 0 gives sqrt(1 + 4/rho^2) (Witt & Mao 1994, cited P:31)."""
    for rho in (0.01, 0.3, 2.0):
        assert abs(single_lens_disk_mu(0.0, rho) - np.sqrt(1 + 4 / rho**2)) < 1e-12 * np.sqrt(1 + 4 / rho**2)


@pytest.mark.parametrize("u,rho", [(0.5, 0.1), (0.05, 0.1), (1.0, 0.01), (0.2, 0.3)])
def test_single_lens_finite_source_limit(u, rho):
    """P-9: q -> 0: the binary code reproduces the uniform-disk single-lens magnification (disk both clear of and
    covering the lens)."""
    s, q = 1.7, 1e-9
    zeta = (0.6 + 0.8j) * u + (-q * s / (1 + q))
    expect = single_lens_disk_mu(u, rho)
    got = mu_ref(s, q, rho, zeta)
    assert abs(got - expect) < 3e-7 * expect, (got, expect)
    # and the paper-style sampler at 1e-6 lands within a few 1e-6
    got2 = api.magnify(_one(s, q, rho, zeta), 1e-6, mode=0)["mu"][0]
    assert abs(got2 - expect) < 5e-6 * expect


def test_large_source_limit():
    """P-11: rho = 50 covers both lenses and all caustics: 3 images everywhere, mu -> sqrt(1+4/rho^2) -> 1."""
    rho = 50.0
    r = api.images_fixed(_one(1.0, 0.3, rho, 0.1 + 0.2j), 512)
    assert np.all(r["count"] == 3)
    got = mu_ref(1.0, 0.3, rho, 0.1 + 0.2j, tol=1e-8)
    assert abs(got - np.sqrt(1 + 4 / rho**2)) < 1e-7
    assert abs(got - 1) < 1e-3


def test_symmetries():
    """P-10: mu(s,q,zeta) = mu(s,q,conj zeta) = mu(s,1/q,-zeta)  (Eq.(1)-(2))."""
    for s, q, rho, zeta in [(1.0, 0.1, 0.1, 0.2 + 0.2j), (0.8, 0.01, 0.02, -0.3 + 0.05j), (2.2, 0.3, 0.05, 1.4 - 0.1j)]:
        a = mu_ref(s, q, rho, zeta)
        b = mu_ref(s, q, rho, np.conj(zeta))
        c = mu_ref(s, 1 / q, rho, -zeta)
        assert abs(a - b) < 2e-7 * a
        assert abs(a - c) < 2e-7 * a, (a, c)


def _bbox(s, q, rho, zeta, pad):
    r = api.images_fixed(_one(s, q, rho, zeta), 2048, prec=1)
    z = r["z"][0][r["kind"][0] != 0]
    return (z.real.min() - pad, z.real.max() + pad, z.imag.min() - pad, z.imag.max() + pad)


@pytest.mark.parametrize("s,q,rho,zeta,ncross", [
    (1.0, 0.1, 0.1, 0.2 + 0.2j, 2),        # Fig.2: two fold crossings
    (1.0, 1.0, 0.05, 0.0 + 0.0j, 0),       # wholly inside the resonant caustic: 5 closed tracks
    (0.8, 0.05, 0.06, -0.03 + 0.0j, None), # covers the central caustic of a close binary (cusps inside the disk)
    (1.6, 0.02, 0.03, 1.0 + 0.01j, None),  # planetary caustic of a wide binary, straddled
])
def test_ray_shooting_agrees(s, q, rho, zeta, ncross):
    """P-12: brute-force inverse ray shooting reproduces the contour-integration area."""
    box = _bbox(s, q, rho, zeta, 0.02)
    nx = int((box[1] - box[0]) / 4e-4) + 1
    ny = int((box[3] - box[2]) / 4e-4) + 1
    rs = api.rayshoot(s, q, rho, zeta, box, nx, ny, sub=32)
    got = mu_ref(s, q, rho, zeta)
    assert abs(got - rs) < 3e-6 * rs, (got, rs)
    if ncross is not None:
        assert api.images_fixed(_one(s, q, rho, zeta), 1024)["ncross"][0] == ncross


def test_fig2_topology_and_crossing_sign():
    """P-6 (tests/golden/fig2_topology.txt): exactly two crossings, one creation and one
    annihilation; with the crossing correction Eq.(11) the fixed-N value converges fast (without it, or with a flipped
    sign, the N = 512 error is > 1e-4 instead of < 1.5e-5).  The sign itself is pinned, separately for creation and
    annihilation, by the fold model in tests/test_oracle_errors.py."""
    rows = [l.split() for l in open(os.path.join(GOLD, "fig2_topology.txt")) if not l.startswith("#")]
    s, q, rho, zr, zi = map(float, rows[0])
    n_cross, n_closed, n_broken, n_pos, n_neg = map(int, rows[1])
    wl = _one(s, q, rho, complex(zr, zi))
    r = api.images_fixed(wl, 256, want_piece=True)
    assert r["ncross"][0] == n_cross
    cnt = r["count"][0]
    # count changes 3->5 once (creation) and 5->3 once (annihilation) going round the boundary
    d = np.diff(np.concatenate([cnt, cnt[:1]]).astype(int))
    assert (d == 2).sum() == 1 and (d == -2).sum() == 1
    # tracks: outside the caustic 1 positive + 2 negative closed tracks (3 complete images); inside, one extra + and
    # one extra - track (the 2 broken tracks): 2 positive and 3 negative tracks in all
    assert n_closed == 3 and n_broken == 2
    assert (r["kind"][0][cnt == 5] > 0).sum(axis=1).max() == n_pos
    assert (r["kind"][0][cnt == 5] < 0).sum(axis=1).max() == n_neg
    truth = mu_ref(s, q, rho, complex(zr, zi))
    assert abs(r["mu"][0] - truth) < 1e-4 * truth
    assert abs(api.images_fixed(wl, 512)["mu"][0] - truth) < 1.5e-5 * truth


def test_parabolic_correction_is_fourth_order():
    """Eq.(9)-(10): with the parabolic correction the fixed-N error falls like N^-4 for a source clear
    of the caustics (the trapezium alone is N^-2) -- pins the 1/24 and 1/12 factors and the sign convention."""
    s, q, rho, zeta = 0.9, 0.2, 0.05, 0.6 + 0.4j
    wl = _one(s, q, rho, zeta)
    truth = mu_ref(s, q, rho, zeta, tol=1e-9)
    err = [abs(api.images_fixed(wl, N, prec=1)["mu"][0] - truth) / truth for N in (16, 32, 64)]
    assert err[0] < 1e-3 and err[2] < 1e-6
    assert 10 < err[0] / err[1] < 24 and 10 < err[1] / err[2] < 24, err
    assert truth > 1.0


def test_positive_tracks_counter_clockwise():
    """S-1: the positive-parity image of a source clear of the caustics is traced counter-clockwise
    as theta increases, the negative ones clockwise; so every parity-weighted track area is positive."""
    s, q, rho, zeta = 0.9, 0.2, 0.05, 0.6 + 0.4j
    r = api.images_fixed(_one(s, q, rho, zeta), 256, prec=1)
    z, kind = r["z"][0], r["kind"][0]
    # follow each real image of sample 0 round the boundary by nearest neighbour
    for k0 in np.where(kind[0] != 0)[0]:
        path, cur = [z[0, k0]], z[0, k0]
        for j in range(1, 256):
            cand = np.where(kind[j] == kind[0, k0])[0]
            k = cand[np.argmin(np.abs(z[j, cand] - cur))]
            cur = z[j, k]
            path.append(cur)
        path = np.array(path + [path[0]])
        signed = 0.5 * np.sum(path[:-1].real * path[1:].imag - path[:-1].imag * path[1:].real)
        assert np.sign(signed) == kind[0, k0]


def test_fig1_zoom_centre():
    """P-5 (tests/golden/fig1_zoom_centre.txt): for the Fig.1 inputs the boundary dips inside the
    planetary-caustic cusp over a tiny theta window and the merging pair sits at the printed zoom centre
    (0.5000595, 0.000535) -- with Im zeta = -0.0035, the mirror image of the text's sign (E-8)."""
    rows = [l.split() for l in open(os.path.join(GOLD, "fig1_zoom_centre.txt")) if not l.startswith("#")]
    s, q, rho, zr, zi = map(float, rows[0])
    cx, cy = map(float, rows[1])
    for sign in (-1, +1):
        zc = complex(zr, sign * zi)
        fine = []
        lo = (2.6215 if sign < 0 else 2 * np.pi - 2.6240)
        for t in np.linspace(lo, lo + 0.0025, 2501):
            p = api.point(s, q, rho, zc, t, 1)
            if p["nreal"] == 5:
                fine.append((t, p))
        assert len(fine) > 10
        width = fine[-1][0] - fine[0][0]
        assert 1.0e-4 < width < 3.0e-4
        # at the first 5-image sample the newly created pair is the two smallest-|J| images
        p = fine[0][1]
        pair = np.argsort(np.abs(p["J"]))[:2]
        zm = p["z"][pair].mean()
        assert abs(zm.real - cx) < 1e-5
        assert abs(zm.imag - (-sign) * cy) < 1e-5 or abs(zm.imag - sign * cy) < 1e-5
        if sign < 0:
            assert abs(zm.imag - cy) < 1e-5          # the printed sign needs Im zeta = -0.0035


def test_fig6_positions_are_smooth():
    """P-7 (tests/golden/fig6_positions.txt): at the two source positions where the paper reports the
    comparison code's spikes the light curve is smooth: paper-style sampler at 1e-4 agrees with the converged
    reference, and with its neighbours."""
    wl = W.fig6_case(n=161, half_width=4e-4)
    a = api.magnify(wl, 1e-4, mode=0)
    b = api.magnify(wl, 1e-6, mode=1, prec=1)
    assert np.all(a["status"] & 1)
    assert np.abs(a["mu"] / b["mu"] - 1).max() < 1e-4        # within the preset tolerance
    curve = b["mu"][2:]
    # no spike: second differences of the converged curve stay small against the curve's own range
    d2 = np.abs(np.diff(curve, 2))
    assert d2.max() < 0.2 * (curve.max() - curve.min())
    xs = wl.zeta[2:, 0]
    for k in (0, 1):
        interp = np.interp(wl.zeta[k, 0], xs, curve)
        assert abs(b["mu"][k] - interp) < 2e-3 * interp


def test_error_estimate_and_stop_rule():
    """when the paper-style sampler stops with E <= tol |A| the true error (vs the extended-precision
    converged reference) is within tol ("all the results are still within the preset relative tolerance"); the cap
    returns value + estimate with status 2."""
    rng = np.random.default_rng(5)
    zs = 0.35 * (rng.uniform(-1, 1, 60) + 1j * rng.uniform(-1, 1, 60))
    wl = W.Workload("t", np.array([1.0]), np.array([0.1]), np.array([0.02]), np.zeros(60, np.int32),
                    np.stack([zs.real, zs.imag], 1).copy(), 1e-4)
    truth = api.magnify(wl, 1e-7, mode=1, prec=1)["mu"]
    for tol in (1e-3, 1e-4, 1e-5):
        r = api.magnify(wl, tol, mode=0)
        assert np.all(r["status"] & 1)
        assert np.all(r["err"] <= tol)
        rel = np.abs(r["mu"] / truth - 1)
        assert rel.max() < tol, (tol, rel.max())
        assert np.median(rel) < 0.1 * tol
    r = api.magnify(wl.subset([0, 1, 2]), 1e-12, mode=0, max_samples=512)
    assert np.all(r["status"] & 2) and np.all(r["nsamples"] <= 512) and np.all(r["nsamples"] > 512 - 64)
    assert np.all(np.isfinite(r["mu"])) and np.all(r["err"] > 1e-12)


def test_adaptive_sampler_concentrates_on_crossings():
    """P:304-312, Fig.4: new samples go where the error is: for the Fig.2 source the added angles are at least
    twice as dense within 0.3 rad of the two caustic crossings (19 % of the circle) as a uniform refinement."""
    wl = W.fig2_case()
    cnt = api.images_fixed(wl, 4096)["count"][0].astype(int)
    th = 2 * np.pi * np.arange(4096) / 4096
    cross = th[np.where(np.diff(np.concatenate([cnt, cnt[:1]])) != 0)[0]]
    t = api.magnify_thetas(1.0, 0.1, 0.1, 0.2 + 0.2j, 1e-5)
    assert len(t) > 128 and np.all(np.diff(t) > 0)
    added = np.array([x for x in t if np.abs(x * 64 / (2 * np.pi) - round(x * 64 / (2 * np.pi))) > 1e-9])
    near = np.min(np.abs(added[:, None] - cross[None, :]), axis=1) < 0.3
    assert near.mean() > 2 * (4 * 0.3) / (2 * np.pi)


def test_slope_detector_rejudging():
    """Slope detector, P:251-268 (reading G-4).  (i) With the default gate it never fires on the worked examples and
    changes nothing.  (ii) Opened up (gate 1e30) at the default 45 degrees it still never fires: real and ghost pairs
    ARE perpendicular across every crossing of these inputs (the geometric fact the detector rests on, Eq.(16)).
    (iii) With the bound tightened to 0 nothing counts as perpendicular: every crossing piece is re-judged pair by
    pair until it is gone ("the whole area piece shall be deleted"): no crossing is left, status bit 32 is
    set, and what remains is the area enclosed by the three image tracks that exist at every theta."""
    wl = W.fig2_case()
    base = api.magnify(wl, 1e-4, mode=0, slope_gate=0.0)
    for gate, cs in ((1e-5, 0.70710678118654752), (1e30, 0.70710678118654752)):
        r = api.magnify(wl, 1e-4, mode=0, slope_gate=gate, slope_cos=cs)
        assert r["mu"][0] == base["mu"][0] and r["nsamples"][0] == base["nsamples"][0] and not (r["status"][0] & 32)
    r = api.magnify(wl, 1e-4, mode=0, slope_gate=1e30, slope_cos=0.0)
    assert r["status"][0] & 32
    assert r["mu"][0] < base["mu"][0] - 0.5          # the merged image's extra lobe (tracks 4 and 5) is gone
    # the long-double twin takes the same decisions
    rl = api.magnify(wl, 1e-4, mode=0, prec=1, slope_gate=1e30, slope_cos=0.0)
    assert abs(rl["mu"][0] / r["mu"][0] - 1) < 1e-9 and rl["nsamples"][0] == r["nsamples"][0]
