"""The five BASELINE.json configs and the paper's worked examples as concrete, seeded arrays."""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Workload:
    """One batch of finite-source magnification problems.

    s, q, rho : float64[n_models]   lens separation, mass ratio, source radius (per model)
    model_id  : int32[n_sources]    model index of every source position
    zeta      : float64[n_sources, 2]  source centres (Re, Im), centre-of-mass frame
    rel_tol   : requested relative accuracy of the magnification (adaptive mode)
    fixed_n   : number of boundary samples in fixed-sampling mode (0 = adaptive config)
    """
    name: str
    s: np.ndarray
    q: np.ndarray
    rho: np.ndarray
    model_id: np.ndarray
    zeta: np.ndarray
    rel_tol: float = 1e-4
    fixed_n: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def n_sources(self) -> int:
        return int(self.zeta.shape[0])

    @property
    def n_models(self) -> int:
        return int(self.s.shape[0])

    def subset(self, idx) -> "Workload":
        """Workload restricted to the source indices `idx` (models are kept whole, ids unchanged)."""
        idx = np.asarray(idx)
        return Workload(self.name + "[subset]", self.s, self.q, self.rho,
                        np.ascontiguousarray(self.model_id[idx]), np.ascontiguousarray(self.zeta[idx]),
                        self.rel_tol, self.fixed_n, dict(self.meta))


def _f64(x):
    return np.ascontiguousarray(np.atleast_1d(np.asarray(x, dtype=np.float64)))


def _pack(zc):
    zc = np.asarray(zc, dtype=np.complex128).ravel()
    return np.ascontiguousarray(np.stack([zc.real, zc.imag], axis=1))


def trajectory(tau, u0, alpha, origin=0.0):
    """zeta(tau) = -(tau + i u0) e^{i alpha} + origin  (complex128 array)."""
    tau = np.asarray(tau, dtype=np.float64)
    return -(tau + 1j * u0) * np.exp(1j * alpha) + origin


def _single_model(name, s, q, rho, zc, rel_tol, fixed_n=0, **meta):
    zeta = _pack(zc)
    return Workload(name, _f64(s), _f64(q), _f64(rho), np.zeros(zeta.shape[0], dtype=np.int32), zeta,
                    rel_tol, fixed_n, meta)


def config1() -> Workload:
    """Single light curve, fixed 256 boundary points: s=1, q=1e-3, rho=1e-3, u0=0.01, alpha=0.5,
    128 epochs tau_k = -1 + 2k/127, primary at origin."""
    s, q, rho = 1.0, 1e-3, 1e-3
    tau = -1.0 + 2.0 * np.arange(128) / 127.0
    z1 = -q * s / (1.0 + q)
    return _single_model("config1", s, q, rho, trajectory(tau, 0.01, 0.5, z1), 1e-4, fixed_n=256)


def config2() -> Workload:
    """Planetary central-caustic-crossing light curve: s=0.9, q=1e-4, rho=1e-3, u0=0.005, alpha=1.2,
    10,000 epochs tau_k = -0.5 + k/9999, primary at origin, adaptive 1e-4."""
    s, q, rho = 0.9, 1e-4, 1e-3
    tau = -0.5 + np.arange(10000) / 9999.0
    z1 = -q * s / (1.0 + q)
    return _single_model("config2", s, q, rho, trajectory(tau, 0.005, 1.2, z1), 1e-4)


def config3(n_models: int = 4096, n_epochs: int = 1000, seed: int = 250103322) -> Workload:
    """MCMC-style parameter batch: n_models lenses x n_epochs epochs tau in [-2, 2], CM frame, tol 1e-4."""
    rng = np.random.default_rng(seed)
    s = np.exp(rng.uniform(np.log(0.3), np.log(3.0), n_models))
    q = np.exp(rng.uniform(np.log(1e-5), 0.0, n_models))
    rho = np.exp(rng.uniform(np.log(1e-4), np.log(1e-2), n_models))
    u0 = rng.uniform(-0.1, 0.1, n_models)
    alpha = rng.uniform(0.0, 2.0 * np.pi, n_models)
    tau = -2.0 + 4.0 * np.arange(n_epochs) / (n_epochs - 1.0)
    zc = trajectory(tau[None, :], u0[:, None], alpha[:, None], 0.0)          # [n_models, n_epochs]
    model_id = np.repeat(np.arange(n_models, dtype=np.int32), n_epochs)
    return Workload("config3", _f64(s), _f64(q), _f64(rho), np.ascontiguousarray(model_id), _pack(zc), 1e-4,
                    meta={"n_models": n_models, "n_epochs": n_epochs, "seed": seed})


def config4(n: int = 1024) -> Workload:
    """Magnification map: n x n cell-centred grid over [-1.5, 1.5]^2, s=1, q=0.1, rho=1e-2, CM frame,
    row-major with y outer, tol 1e-4."""
    x = -1.5 + 3.0 * (np.arange(n) + 0.5) / n
    zc = x[None, :] + 1j * x[:, None]
    return _single_model("config4", 1.0, 0.1, 1e-2, zc, 1e-4, grid=n)


def config5(n: int = 100000, seed: int = 250103323) -> Workload:
    """High-accuracy stress: n sources each with its own lens; first half close binaries s in U(0.2,0.5),
    second half wide s in U(2,4); q log-uniform [1e-6,1]; rho log-uniform [1e-3,1e-1]; zeta uniform in
    [-1,1]^2; CM frame; tol 1e-6."""
    rng = np.random.default_rng(seed)
    h = n // 2
    s = np.concatenate([rng.uniform(0.2, 0.5, h), rng.uniform(2.0, 4.0, n - h)])
    q = np.exp(rng.uniform(np.log(1e-6), 0.0, n))
    rho = np.exp(rng.uniform(np.log(1e-3), np.log(1e-1), n))
    re = rng.uniform(-1.0, 1.0, n)
    im = rng.uniform(-1.0, 1.0, n)
    return Workload("config5", _f64(s), _f64(q), _f64(rho), np.arange(n, dtype=np.int32), _pack(re + 1j * im),
                    1e-6, meta={"seed": seed})


def fig2_case() -> Workload:
    """PAPER.md:159 (Fig. 2): s=1, q=0.1, rho=0.1, zeta=0.2+0.2i; boundary crosses the caustic twice."""
    return _single_model("fig2", 1.0, 0.1, 0.1, [0.2 + 0.2j], 1e-4, fixed_n=256)


def fig1_case(mirror: bool = True) -> Workload:
    """PAPER.md:118 (Fig. 1): s=0.5, q=1e-6, rho=1e-4, zeta=-1.49981640625 +/- 0.0035i.  mirror=True takes
    Im zeta = -0.0035 (the sign that reproduces the printed zoom centre, reading E-8)."""
    im = -0.0035 if mirror else 0.0035
    return _single_model("fig1", 0.5, 1e-6, 1e-4, [-1.49981640625 + 1j * im], 1e-4, fixed_n=256)


def fig6_case(n: int = 201, half_width: float = 4e-4) -> Workload:
    """PAPER.md:362-364 (Fig. 6): s=0.5, q=1e-6, rho=1e-4, theta_y=-0.0035; a light-curve segment of n
    epochs centred between the two positions where the paper reports the comparison code spikes
    (theta_x=-1.49998960 and -1.49993410), which are included exactly as the first two entries."""
    xs = np.concatenate([[-1.49998960, -1.49993410],
                         -1.4999618 + half_width * np.linspace(-1.0, 1.0, n)])
    return _single_model("fig6", 0.5, 1e-6, 1e-4, xs - 0.0035j, 1e-4)


# ---------------------------------------------------------------------------------------------------------
# Second workload family: the paper's own caustic-dense test inputs.  Window extents are
# figure-only in the paper (not in its text); the ones below are this repo's choice and are stated here.
# ---------------------------------------------------------------------------------------------------------
_FIG5 = {
    # name: (s, q, rho, origin of the map = position of the planetary / resonant caustic, half-width in x)
    "close": (0.5, 1e-4, 5e-5, -1.5 + 0.035j, 4e-3),
    "resonant": (1.0, 1e-4, 1e-3, 0.0 + 0.0j, 0.12),
    "wide": (3.0, 1e-4, 1e-4, 2.666 + 0.0j, 8e-3),
}


def fig5_map(case: str = "close", nx: int = 480, ny: int = 340) -> Workload:
    """PAPER.md:342, P:352 (Fig. 5): source-plane map of nx x ny = 480 x 340 extended sources over the planetary
    (s = 0.5, 3) or resonant (s = 1) caustic, q = 1e-4, rho matched to the caustic, tol 1e-4.  Cell-centred grid,
    row-major with y outer, centred on the origin the caption gives; half-width in x as tabulated above (about twice
    the caustic), half-width in y = half-width in x * ny / nx."""
    s, q, rho, o, hx = _FIG5[case]
    hy = hx * ny / nx
    x = o.real - hx + 2.0 * hx * (np.arange(nx) + 0.5) / nx
    y = o.imag - hy + 2.0 * hy * (np.arange(ny) + 0.5) / ny
    return _single_model("fig5_" + case, s, q, rho, x[None, :] + 1j * y[:, None], 1e-4, nx=nx, ny=ny)


def _planetary_caustic(s, q):
    """Centre and linear scale of the planetary caustic (textbook perturbative expressions, used only to PLACE
    source grids): on the axis at s - 1/s for wide binaries, off the axis by 2 sqrt(q (1 - s^2)) / s for close ones;
    scale ~ sqrt(q) s^3 (close), sqrt(q) / s^2 (wide), never more than the resonant size ~ q^(1/3)."""
    xc = s - 1.0 / s
    yc = np.where(s < 1.0, 2.0 * np.sqrt(q * np.maximum(1.0 - s * s, 0.0)) / s, 0.0)
    scale = np.where(s < 1.0, np.sqrt(q) * s ** 3, np.sqrt(q) / s ** 2)
    return xc + 1j * yc, np.minimum(4.0 * scale, 1.5 * q ** (1.0 / 3.0))


def fig7_grid(n_s: int = 16, n_q: int = 12, n_side: int = 30, rho: float = 1e-4) -> Workload:
    """PAPER.md:368 (Fig. 7): parameter-space sweep.  n_s x n_q lenses, s linear in [0.5, 3], q log-spaced in
    [1e-6, 1e-2]; each with an n_side x n_side = 30 x 30 cell-centred grid of sources of radius rho = 1e-4 covering
    the planetary (resonant) caustic: centred on it, half-width max(2 x caustic scale, 10 rho).  tol 1e-4."""
    sv = np.linspace(0.5, 3.0, n_s)
    qv = np.exp(np.linspace(np.log(1e-6), np.log(1e-2), n_q))
    S, Q = [a.ravel() for a in np.meshgrid(sv, qv, indexing="ij")]
    c, scale = _planetary_caustic(S, Q)
    hw = np.maximum(2.0 * scale, 10.0 * rho)
    u = -1.0 + 2.0 * (np.arange(n_side) + 0.5) / n_side
    g = (u[None, :] + 1j * u[:, None]).ravel()                          # [n_side^2]
    zc = c[:, None] + hw[:, None] * g[None, :]
    n_m = S.size
    model_id = np.repeat(np.arange(n_m, dtype=np.int32), n_side * n_side)
    return Workload("fig7_grid", _f64(S), _f64(Q), _f64(np.full(n_m, rho)), np.ascontiguousarray(model_id), _pack(zc),
                    1e-4, meta={"n_s": n_s, "n_q": n_q, "n_side": n_side})


def lowq_sweep(n: int = 4000, seed: int = 250103324) -> Workload:
    """Low-mass-ratio robustness sweep over the validated domain of P:374 (0.1 <= s <= 10, q >= 1e-9): n sources,
    each with its own lens: s log-uniform in [0.1, 10], q log-uniform in [1e-9, 1e-6], rho log-uniform in
    [1e-4, 1e-2]; the source centre is drawn uniformly in a square of half-width 3 max(rho, caustic scale) around
    the planetary caustic, so most disks touch or cover it.  tol 1e-4."""
    rng = np.random.default_rng(seed)
    s = np.exp(rng.uniform(np.log(0.1), np.log(10.0), n))
    q = np.exp(rng.uniform(np.log(1e-9), np.log(1e-6), n))
    rho = np.exp(rng.uniform(np.log(1e-4), np.log(1e-2), n))
    c, scale = _planetary_caustic(s, q)
    hw = 3.0 * np.maximum(rho, scale)
    zc = c + hw * (rng.uniform(-1.0, 1.0, n) + 1j * rng.uniform(-1.0, 1.0, n))
    return Workload("lowq_sweep", _f64(s), _f64(q), _f64(rho), np.arange(n, dtype=np.int32), _pack(zc), 1e-4,
                    meta={"seed": seed})


def domain_corners(n: int = 4000, seed: int = 250103325) -> Workload:
    """The corners of the validated domain of P:374: s uniform in [0.1, 0.2] or [5, 10] (half each), q log-uniform in
    [1e-9, 1e-7], rho log-uniform in [1e-4, 1e-2]; source centre within 3 rho of the planetary-caustic position
    s - 1/s on the axis.  tol 1e-4."""
    rng = np.random.default_rng(seed)
    s = np.where(rng.random(n) < 0.5, rng.uniform(0.1, 0.2, n), rng.uniform(5.0, 10.0, n))
    q = np.exp(rng.uniform(np.log(1e-9), np.log(1e-7), n))
    rho = np.exp(rng.uniform(np.log(1e-4), np.log(1e-2), n))
    zc = (s - 1.0 / s) + 3.0 * rho * (rng.uniform(-1.0, 1.0, n) + 1j * rng.uniform(-1.0, 1.0, n))
    return Workload("domain_corners", _f64(s), _f64(q), _f64(rho), np.arange(n, dtype=np.int32), _pack(zc), 1e-4,
                    meta={"seed": seed})


def get(name: str, **kw) -> Workload:
    table = {"config1": config1, "config2": config2, "config3": config3, "config4": config4,
             "config5": config5, "fig1": fig1_case, "fig2": fig2_case, "fig6": fig6_case, "fig5_map": fig5_map,
             "fig7_grid": fig7_grid, "lowq_sweep": lowq_sweep, "domain_corners": domain_corners}
    return table[name](**kw)
