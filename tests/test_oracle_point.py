"""Pins of the oracle's per-sample quantities (T-3..T-5) against what the
paper and the mathematics fix -- all expected values are computed here from Eq.(1)/(2)/(7) directly."""
import numpy as np
import pytest

from oracle import api


def lens(s, q):
    return 1 / (1 + q), q / (1 + q), -q * s / (1 + q), s / (1 + q)


def lens_eq_residual(s, q, zeta, z):
    """zeta - [z + m1/(conj z1 - conj z) + m2/(conj z2 - conj z)], Eq.(1), CM frame."""
    m1, m2, z1, z2 = lens(s, q)
    return zeta - (z + m1 / np.conj(z1 - z) + m2 / np.conj(z2 - z))


def fprime(s, q, z):
    m1, m2, z1, z2 = lens(s, q)
    return m1 / (z1 - z) ** 2 + m2 / (z2 - z) ** 2


def random_cases(n, seed, qmin=1e-7):
    rng = np.random.default_rng(seed)
    for _ in range(n):
        s = np.exp(rng.uniform(np.log(0.3), np.log(3)))
        q = np.exp(rng.uniform(np.log(qmin), 0))
        zc = rng.uniform(-1.5, 1.5) + 1j * rng.uniform(-1.5, 1.5)
        if rng.uniform() < 0.3:          # resonant binaries probed near the centre: inside the caustic, 5 images
            s, q = rng.uniform(0.8, 1.3), max(q, rng.uniform(0.05, 1.0))
            zc = 0.25 * (rng.uniform(-1, 1) + 1j * rng.uniform(-1, 1))
        rho = 10 ** rng.uniform(-4, -1)
        th = rng.uniform(0, 2 * np.pi)
        yield s, q, rho, zc, th


@pytest.mark.parametrize("prec", [0, 1])
def test_images_satisfy_lens_equation_counts_and_parity(prec):
    """P-3: real images satisfy Eq.(1); 3 or 5 of them; parity sum -1; J sign is the parity (Eq.7)."""
    n5 = 0
    for s, q, rho, zc, th in random_cases(400, 3):
        p = api.point(s, q, rho, zc, th, prec)
        zeta = zc + rho * np.exp(1j * th)
        real = p["kind"] != 0
        assert p["nreal"] in (3, 5) and real.sum() == p["nreal"]
        assert p["kind"][real].sum() == -1
        res = lens_eq_residual(s, q, zeta, p["z"][real])
        # a position error dz shows up as ~(1+|f'|) dz in Eq.(1): tiny images next to the planet have |f'| >> 1
        cond = 1 + np.abs(fprime(s, q, p["z"][real]))
        assert np.all(np.abs(res) < 1e-11 * cond), (s, q, zeta, res, cond)
        if not p["repaired"]:
            Jd = 1 - np.abs(fprime(s, q, p["z"][real])) ** 2
            assert np.all(np.sign(Jd) == p["kind"][real])
        # ghosts do NOT satisfy Eq.(1)
        if p["nreal"] == 3:
            assert np.abs(lens_eq_residual(s, q, zeta, p["z"][~real])).min() > 1e-7
        n5 += p["nreal"] == 5
    assert n5 > 5          # both cases exercised


def test_known_image_counts():
    """a point source inside a caustic has 5 images, outside 3.  Equal-mass s=1 binary: zeta=0 is inside
    the resonant caustic; zeta=3+2i is far outside."""
    assert api.point(1.0, 1.0, 1e-3, 0.0, 0.3)["nreal"] == 5
    assert api.point(1.0, 1.0, 1e-3, 3 + 2j, 0.3)["nreal"] == 3


@pytest.mark.parametrize("prec", [0, 1])
def test_sum_of_residuals_is_zero(prec):
    """T-3, Eq.(13)-(14): the five residuals sum to zero."""
    for s, q, rho, zc, th in random_cases(200, 5):
        p = api.point(s, q, rho, zc, th, prec)
        assert abs(p["R"].sum()) < 1e-11 * max(1.0, np.abs(p["R"]).max())


def test_residual_matches_eq12_in_cm_frame():
    """Eq.(12) evaluated here in the CM frame equals the oracle's (planet-frame) residual (Eq.15)."""
    for s, q, rho, zc, th in random_cases(50, 6, qmin=1e-3):
        p = api.point(s, q, rho, zc, th, 1)
        zeta = zc + rho * np.exp(1j * th)
        m1, m2, z1, z2 = lens(s, q)
        R = zeta - p["z"] + m1 / np.conj(p["z"] - z1) + m2 / np.conj(p["z"] - z2)
        assert np.abs(R - p["R"]).max() < 1e-10


def test_ghost_pair_geometry():
    """T-5 / P-13: a ghost pair has opposite residuals of equal length, equal to the pair separation."""
    seen = 0
    for s, q, rho, zc, th in random_cases(300, 8):
        p = api.point(s, q, rho, zc, th, 1)
        g = np.where(p["kind"] == 0)[0]
        assert len(g) in (0, 2)
        if len(g) == 2:
            a, b = g
            Ra, Rb = p["R"][a], p["R"][b]
            sep = p["z"][b] - p["z"][a]
            assert abs(Ra + Rb) < 1e-9 * abs(Ra)
            assert abs(Ra - sep) < 1e-9 * abs(Ra)
            seen += 1
    assert seen > 100


def test_generalised_point_magnification_sum():
    """T-4 / P-4: sum over all five roots of 1/(1 - f'(z_k) f'(w_k)) = 1 with conj(w_k) = conj(zeta) - f(z_k)...
    written with w_k = conj(zeta) - f(z_k) evaluated through f' on the real-axis lens pair; for 5 real images
    this is the classical sum of signed magnifications sum p/|J| = 1."""
    n5 = 0
    for s, q, rho, zc, th in random_cases(300, 9, qmin=1e-4):
        p = api.point(s, q, rho, zc, th, 1)
        zeta = zc + rho * np.exp(1j * th)
        m1, m2, z1, z2 = lens(s, q)
        z = p["z"]
        f = m1 / (z1 - z) + m2 / (z2 - z)
        w = np.conj(zeta) - f
        tot = np.sum(1 / (1 - fprime(s, q, z) * fprime(s, q, w)))
        assert abs(tot - 1) < 1e-8, (s, q, zeta, tot)
        if p["nreal"] == 5:
            n5 += 1
            assert abs(np.sum(p["kind"] / np.abs(p["J"])) - 1) < 1e-8
            assert abs(np.sum(1 / p["J"]) - 1) < 1e-8      # pins the oracle's own J
    assert n5 > 5


def test_paczynski_limit_point_source():
    """P-8: q -> 0 (and separately s -> infinity): sum 1/|J| over real images -> (u^2+2)/(u sqrt(u^2+4))."""
    for u in (0.1, 0.5, 1.3):
        zeta = 0.6 * u + 0.8j * u
        # q -> 0: the whole mass sits at z1 ~ 0
        s, q = 1.7, 1e-12
        p = api.point(s, q, 1e-9, zeta, 0.0, 0)
        real = p["kind"] != 0
        uu = abs(zeta + 1e-9 - (-q * s / (1 + q)))
        A = np.sum(1 / np.abs(p["J"][real]))
        assert abs(A - (uu**2 + 2) / (uu * np.sqrt(uu**2 + 4))) < 1e-8
        # s -> infinity with q = 1: lens 1 alone has mass 1/2, Einstein radius sqrt(1/2); companion shear ~ m2/s^2
        s, q = 2000.0, 1.0
        z1 = -q * s / (1 + q)
        # the far lens adds the constant deflection m2/s (Eq.1 at |z - z2| ~ s); what is left is its shear m2/s^2
        # (long double face: at s >> 10, outside P:374's domain, the FP64 quintic is ill-conditioned near the far lens)
        p = api.point(s, q, 1e-9, z1 + zeta * np.sqrt(0.5) + 0.5 / s, 0.0, 1)
        real = p["kind"] != 0
        J = p["J"][real]
        near = np.abs(p["z"][real] - z1) < 10      # the third image sits next to the far lens with ~0 flux
        A = np.sum(1 / np.abs(J[near]))
        assert abs(A - (u**2 + 2) / (u * np.sqrt(u**2 + 4))) < 1e-5


def _track(s, q, rho, zc, th, h):
    """The five roots at th-h, th, th+h (long double face), matched to the middle sample by nearest neighbour."""
    mid = api.point(s, q, rho, zc, th, 1)
    out = []
    for t in (th - h, th + h):
        p = api.point(s, q, rho, zc, t, 1)
        idx = [int(np.argmin(np.abs(p["z"] - z))) for z in mid["z"]]
        out.append(p["z"][idx])
    return mid, out[0], out[1]


def test_zprime_and_wedge_against_finite_differences():
    """Eq.(10) as repaired (E-2, E-3): z' and z'^z'' of every real image equal central finite
    differences of the tracked image position (independent of any formula for f', f'')."""
    rng = np.random.default_rng(21)
    checked = 0
    for s, q, rho, zc, th in random_cases(60, 22, qmin=1e-3):
        rho = max(rho, 1e-2)
        h = 2e-4
        mid, lo, hi = _track(s, q, rho, zc, th, h)
        for k in range(5):
            if mid["kind"][k] == 0 or abs(mid["J"][k]) < 0.05:
                continue
            d1 = (hi[k] - lo[k]) / (2 * h)
            d2 = (hi[k] - 2 * mid["z"][k] + lo[k]) / h**2
            scale = abs(d1) + 1e-30
            assert abs(mid["zp"][k] - d1) < 2e-5 * scale, (s, q, zc, th, k)
            wfd = d1.real * d2.imag - d1.imag * d2.real
            wscale = abs(d1) * abs(d2) + 1e-30
            assert abs(mid["w"][k] - wfd) < 1e-3 * wscale + 1e-12, (s, q, zc, th, k, mid["w"][k], wfd)
            checked += 1
    assert checked > 100


def test_double_and_long_double_classify_alike():
    """The 2-cycle test is threshold-free (G-1): FP64 and extended precision give the same kinds on
    generic inputs, including q = 1e-7."""
    for s, q, rho, zc, th in random_cases(500, 31):
        a, b = api.point(s, q, rho, zc, th, 0), api.point(s, q, rho, zc, th, 1)
        ia = [int(np.argmin(np.abs(a["z"] - z))) for z in b["z"]]
        assert sorted(ia) == [0, 1, 2, 3, 4]
        assert np.all(a["kind"][ia] == b["kind"])
        assert np.abs(a["z"][ia] - b["z"]).max() < 1e-9


def test_paper_workload_generators_shapes():
    """SURVEY 8(f) N2/N3 inputs: shapes and placement as documented (Fig. 5: 480 x 340 maps centred on the origins
    the caption prints; Fig. 7: 30 x 30 sources per lens; low-q sweep inside P:374's domain)."""
    import workloads as W
    m = W.fig5_map("close")
    assert m.n_sources == 480 * 340 and m.n_models == 1 and m.rho[0] == 5e-5
    assert abs(m.zeta[:, 0].mean() + 1.5) < 1e-12 and abs(m.zeta[:, 1].mean() - 0.035) < 1e-12
    assert abs(W.fig5_map("wide").zeta[:, 0].mean() - 2.666) < 1e-12
    g = W.fig7_grid()
    assert g.n_sources == g.n_models * 900 and g.s.min() == 0.5 and g.s.max() == 3.0
    assert abs(g.q.min() - 1e-6) < 1e-18 and abs(g.q.max() - 1e-2) < 1e-12 and np.all(g.rho == 1e-4)
    lo = W.lowq_sweep()
    assert lo.q.min() >= 1e-9 and lo.q.max() <= 1e-6 and lo.s.min() >= 0.1 and lo.s.max() <= 10.0
    # the oracle finds caustic crossings in a sample of the low-q sweep (the placement does its job)
    sub = lo.subset(np.arange(0, lo.n_sources, 40))
    r = api.magnify(sub, 1e-4, mode=0)
    assert (r["nsamples"] > 64).mean() > 0.05 and np.all(r["status"] & 1)
