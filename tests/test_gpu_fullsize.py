"""Full-size acceptance (-m gpu): every BASELINE config and the paper's own maps at their full sizes, the CUDA path
through the C ABI against the oracle's converged reference (mode 1: 256 uniform samples, bisection of the worst eighth
until the estimate is below a tenth of 1e-6), source by source.

  * north_star bar: both sides at target 1e-6  ->  |mu_gpu - mu_ref| / mu_ref <= 1e-5 at EVERY source;
  * the paper's claim ("all the results are still within the preset relative tolerance of 1e-4"): the CUDA path at
    its working tolerance 1e-4 against the same reference  ->  within 1e-4, with the exceptions DESIGN.md section 2
    (reading L-4) documents and this file counts.

Oracle cost (OpenMP, all host cores; measured on the 8-core build box): ~0.65 ms per source for the reference, i.e.
~2 min for a 163,200-source map, ~11 min for config 4 -- about half of that on the GPU box's 16 cores.  Config 3 is
checked on a seeded 1 % subsample (40,960 sources; SURVEY 8(d) allows it when the full oracle run exceeds ~10 min:
4.1 M sources would take ~45 min); everything else is complete.
"""
import numpy as np
import pytest

import workloads as W
from oracle import api

pytestmark = pytest.mark.gpu

MU_TOL = 1e-5          # north_star: both paths at target 1e-6


@pytest.fixture(scope="module")
def ctx():
    import paper_2501_03322_b200 as P
    c = P.Context(1 << 21)
    yield c
    c.close()


def _check(ctx, wl, allow_beyond_tol=0, worst_allowed=1e-4):
    ref = api.magnify(wl, 1e-6, mode=1, prec=0)
    assert np.all(ref["status"] & 1)
    g6 = ctx.magnify_workload(wl, 1e-6)
    st6 = ctx.twk_last_stats()
    rel6 = np.abs(g6["mu"] / ref["mu"] - 1)
    assert np.all(np.isfinite(g6["mu"]))
    assert rel6.max() <= MU_TOL, (wl.name, rel6.max(), int(np.argmax(rel6)))
    g4 = ctx.magnify_workload(wl, 1e-4)
    rel4 = np.abs(g4["mu"] / ref["mu"] - 1)
    st = g4["status"].astype(np.uint32)
    assert np.all(st & 1), "every source converges at 1e-4"
    n_bad = int((rel4 > 1e-4).sum())
    assert n_bad <= allow_beyond_tol and rel4.max() <= worst_allowed, (wl.name, n_bad, rel4.max(), np.argsort(-rel4)[:5])
    print(f"{wl.name}: n={wl.n_sources} at 1e-6 max {rel6.max():.2e} (stage2 {st6['n_stage2']}, stage3 {st6['n_stage3']}); "
          f"at 1e-4 max {rel4.max():.2e}, beyond tol {n_bad}, mean samples {g4['nsamples'].mean():.1f}")
    return g6, g4, ref, st6


@pytest.mark.parametrize("case", ["resonant", "wide"])
def test_fig5_maps_complete(ctx, case):
    """P:342-344, Fig.5: the 480 x 340 source-plane maps (q = 1e-4), every source."""
    _check(ctx, W.fig5_map(case))


def test_fig5_close_map_complete(ctx):
    """The close-binary map (s = 0.5, rho = 5e-5): 163,200 sources.  Reading L-4: a boundary that dips into
    the caustic and out again BETWEEN two adjacent samples of the first 64 leaves no trace at the interval's end points;
    one source of this map does (5.6e-4 off at 1e-4), two more sit at 1.2e-4 (crossing piece next to a cusp).  At most
    that many; at 1e-6 everything is within the bar."""
    _check(ctx, W.fig5_map("close"), allow_beyond_tol=4, worst_allowed=6e-4)


def test_fig7_grid_complete(ctx):
    """P:368, Fig.7: 16 x 12 lenses over (s, q) in [0.5, 3] x [1e-6, 1e-2], 30 x 30 sources each: 172,800 sources."""
    _check(ctx, W.fig7_grid())


def test_config4_complete(ctx):
    """BASELINE config 4: the full 1024 x 1024 map (1,048,576 sources).  Two of them (a mirror pair at
    zeta = -0.1509 +- 0.3062i) hide a double crossing between two of the first 64 samples (reading L-4): 1.9e-4 off at
    tol 1e-4; at 1e-6 every source is within the bar."""
    g6, g4, ref, st6 = _check(ctx, W.config4(), allow_beyond_tol=2, worst_allowed=2.5e-4)
    assert st6["n_stage3"] > 0                      # the 4096-sample stage ran at 1e-6


def test_config5_complete(ctx):
    """BASELINE config 5: all 100,000 sources at its own tolerance 1e-6."""
    wl = W.config5()
    ref = api.magnify(wl, 1e-6, mode=1, prec=0)
    g = ctx.magnify_workload(wl, 1e-6)
    rel = np.abs(g["mu"] / ref["mu"] - 1)
    assert np.all(np.isfinite(g["mu"])) and rel.max() <= MU_TOL, (rel.max(), int(np.argmax(rel)))
    assert np.all(g["status"].astype(np.uint32) & 1)


def test_config3_one_percent(ctx):
    """BASELINE config 3: a seeded 1 % subsample (40,960 of 4,096,000 sources) source by source; the full batch in one
    call (the launch configuration bench.py times) must give the same values at those sources."""
    import paper_2501_03322_b200 as P
    full = W.config3()
    idx = np.sort(np.random.default_rng(2501).choice(full.n_sources, 40960, replace=False))
    g6, g4, ref, _ = _check(ctx, full.subset(idx))
    c = P.Context(full.n_sources)
    whole = c.magnify_workload(full, 1e-4)
    c.close()
    assert np.all(np.isfinite(whole["mu"])) and np.all(whole["mu"] >= 1.0 - 1e-6)
    d = np.abs(whole["mu"][idx] / g4["mu"] - 1)
    # same arithmetic; a source may take the hand-over or the recompute route depending on the batch around it
    assert np.median(d) < 1e-13 and d.max() < 2e-6


@pytest.mark.parametrize("family", ["lowq", "corners", "config5", "config3"])
def test_fresh_seed_campaign(ctx, family):
    """Seeds no other test uses: 30,000 sources of the low-q sweep (q down to 1e-9 next to the planetary caustic), 20,000
    at the corners of the validated domain, 20,000 fresh config-5 draws and 40,000 epochs of fresh config-3 light
    curves, source by source against the oracle's converged reference: within 1e-5 at target 1e-6 (north_star), and at
    the working tolerance 1e-4 within the tolerance except for at most a few sources in 10,000 (the L-4 cases and the
    crossing pieces next to a cusp that DESIGN.md documents), never more than 5 tolerances away."""
    if family == "lowq":
        wl = W.lowq_sweep(n=30000, seed=250103401)
    elif family == "corners":
        wl = W.domain_corners(n=20000, seed=250103402)
    elif family == "config5":
        wl = W.config5(n=20000, seed=250103403)
    else:
        wl = W.config3(n_models=40, n_epochs=1000, seed=250103404)
    ref = api.magnify(wl, 1e-6, mode=1, prec=0)
    assert np.all(ref["status"] & 1)
    g6 = ctx.magnify_workload(wl, 1e-6)
    rel6 = np.abs(g6["mu"] / ref["mu"] - 1)
    assert np.all(np.isfinite(g6["mu"])) and rel6.max() <= MU_TOL, (family, rel6.max(), int(np.argmax(rel6)))
    g4 = ctx.magnify_workload(wl, 1e-4)
    rel4 = np.abs(g4["mu"] / ref["mu"] - 1)
    assert np.all(g4["status"].astype(np.uint32) & 1)
    assert (rel4 > 1e-4).sum() <= max(1, wl.n_sources // 5000) and rel4.max() < 5e-4, (family, (rel4 > 1e-4).sum(), rel4.max())
    print(f"{family}: n={wl.n_sources} at 1e-6 max {rel6.max():.2e}; at 1e-4 max {rel4.max():.2e}, beyond tol {(rel4 > 1e-4).sum()}")


def test_config2_complete(ctx):
    _check(ctx, W.config2())


def test_cap_4096_like_for_like(ctx):
    """The real sample cap: at tol 1e-12 the Fig.1 / Fig.2 sources and a central-caustic source run into
    4096 samples in the third stage; value, estimate, count and status match the oracle's paper-style sampler."""
    for wl in (W.fig2_case(), W.fig1_case(), W.config2().subset([5003])):
        g = ctx.magnify_workload(wl, 1e-12)
        st = ctx.twk_last_stats()
        o = api.magnify(wl, 1e-12, mode=0)
        assert st["n_stage3"] == 1
        assert int(g["status"][0]) & 2 and o["status"][0] & 2
        assert g["nsamples"][0] == o["nsamples"][0] and 4096 - 64 < g["nsamples"][0] <= 4096
        # (at 4096 samples the estimate ~1e-9 sits on rounding-level ties of the sampler: same size, not same digits)
        assert abs(g["mu"][0] / o["mu"][0] - 1) < 1e-9 and 0.5 < g["err"][0] / o["err"][0] < 2.0


def test_hidden_crossing_guard_closes_the_l4_cases():
    """Option hidden_crossing_guard = 1 (reading L-4, an extension): like-for-like with the oracle's guard, and on the two
    complete maps that hold the known L-4 sources no source is left beyond the tolerance because of a hidden crossing
    (what remains on the close map are the two crossing pieces next to a cusp at 1.2e-4)."""
    import paper_2501_03322_b200 as P
    c = P.Context(1 << 21, hidden_crossing_guard=1)
    for name, worst in (("close", 1.3e-4), ):
        wl = W.fig5_map(name)
        ref = api.magnify(wl, 1e-6, mode=1, prec=0)
        g = c.magnify_workload(wl, 1e-4)
        rel = np.abs(g["mu"] / ref["mu"] - 1)
        assert (rel > 1e-4).sum() <= 2 and rel.max() < worst, (name, (rel > 1e-4).sum(), rel.max())
    full = W.config4()
    zc = full.zeta[:, 0] + 1j * full.zeta[:, 1]
    near = np.where(np.abs(np.abs(zc) - 0.34) < 0.05)[0]                    # the ring of the map that holds the two L-4 sources
    wl = full.subset(near)
    assert np.any(np.abs(zc[near] - (-0.15087891 + 0.30615234j)) < 1e-6)
    ref = api.magnify(wl, 1e-6, mode=1, prec=0)
    g = c.magnify_workload(wl, 1e-4)
    assert np.abs(g["mu"] / ref["mu"] - 1).max() <= 1e-4
    # like-for-like with the oracle's guard: same sample counts, same values
    for wl in (W.fig5_map("close").subset(np.arange(60000, 90000, 7)), W.config4().subset(near[::5])):
        g = c.magnify_workload(wl, 1e-4)
        o = api.magnify(wl, 1e-4, mode=0, hidden_guard=1)
        same = g["nsamples"] == o["nsamples"]
        assert same.mean() > 0.97 and np.quantile(np.abs(g["mu"] / o["mu"] - 1)[same], 0.99) < 1e-8
        assert np.abs(g["mu"] / o["mu"] - 1).max() < 1e-4
    c.close()
