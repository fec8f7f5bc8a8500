"""GPU parity (-m gpu): twk_magnify at ragged batch sizes under every combination of the context options, on five lens
families that the BASELINE configs do not reach (sources larger than the Einstein ring, q > 1, sources hugging the
central caustic of a planet, the resonant regime, the whole validated domain of P:374), against the oracle.

Seeded; the draws below come from the test's own generator, no value is stored.  What must hold for every trial:
  * the same sources are finite / NaN on both sides, the sample count never exceeds the cap, status has exactly one of
    'converged' (1) and 'cap' (2);
  * a source that needed only the first iteration (64 uniform samples) on both sides has the oracle's value to
    rounding (identical samples, identical formulas; 1e-7: the area of a source of radius 1e-5 at |z| ~ 1 is a sum
    with ten digits of cancellation);
  * against the oracle's converged reference (mode 1 at 1e-7): every source the CUDA path reports as converged is
    within 1.5 rel_tol and at most 0.2 % of them are beyond rel_tol (Eq.(17)-(18) is an estimate, not a bound: the
    largest excess seen in 5,000 further trials of this generator was 1.4 tol on a resonant-caustic source -- apart from
    one hidden double crossing, reading L-4, 59 tol at tol 1e-5, identical in the oracle's sampler and closed
    by the hidden_crossing_guard option; the seeds below contain none);
  * a source that hit the cap returns a finite value and an estimate above the tolerance (value and estimated
    error are returned; at a cap of 64 samples the value is the oracle's by the rule above, and how far a source that was
    stopped early is from the truth is not a property the method promises).
"""
import numpy as np
import pytest

import workloads as W
from oracle import api

pytestmark = pytest.mark.gpu

SIZES = [1, 2, 3, 4, 5, 31, 32, 33, 63, 64, 65, 127, 128, 129, 255, 257, 1000, 3553]
FAMILIES = ["domain", "big_source", "q_above_1", "central_caustic", "resonant"]


def _draw(rng, n, fam):
    lu = lambda a, b: np.exp(rng.uniform(np.log(a), np.log(b), n))
    if fam == "domain":            # 0.1 <= s <= 10, q >= 1e-9
        s, q, rho, z = lu(0.1, 10), lu(1e-9, 1), lu(1e-5, 0.3), rng.uniform(-2, 2, (n, 2))
    elif fam == "big_source":      # rho up to five Einstein radii
        s, q, rho, z = lu(0.3, 3), lu(1e-4, 1), lu(0.1, 5), rng.uniform(-1, 1, (n, 2))
    elif fam == "q_above_1":       # the mass-swapped system (accepted)
        s, q, rho, z = lu(0.3, 3), lu(1, 1e4), lu(1e-3, 1e-1), rng.uniform(-1.5, 1.5, (n, 2))
    elif fam == "central_caustic":
        s, q, rho = lu(0.5, 2), lu(1e-4, 1e-1), lu(1e-4, 1e-2)
        z1 = -q * s / (1 + q)
        z = np.stack([z1 + rng.normal(0, 0.15, n) * np.sqrt(q), rng.normal(0, 0.15, n) * np.sqrt(q)], 1)
    else:                          # resonant
        s, q, rho, z = rng.uniform(0.8, 1.25, n), lu(1e-3, 1), lu(1e-3, 5e-2), rng.uniform(-0.6, 0.6, (n, 2))
    return s, q, rho, np.ascontiguousarray(z)


def _trials(seed, count):
    rng = np.random.default_rng(seed)
    for k in range(count):
        n = int(rng.choice(SIZES))
        fam = FAMILIES[k % len(FAMILIES)]
        tol = float(rng.choice([1e-3, 1e-4, 1e-5, 1e-6]))
        opts = dict(max_samples=int(rng.choice([64, 128, 192, 512, 576, 1024, 4096])),
                    handoff_slots=int(rng.choice([-1, 0, 1, 5, 64])), subtract_avg_tol=int(rng.choice([1, 1, 0])))
        shared = rng.random() < 0.25           # one lens for the whole batch
        s, q, rho, z = _draw(rng, 1 if shared else n, fam)
        if shared:
            z = _draw(rng, n, fam)[3]
        explicit_ids = shared or rng.random() < 0.5      # model_id given, or NULL with n_models == n_sources
        if shared and rng.random() < 0.5:
            explicit_ids = False                         # NULL with n_models == 1
        mid = np.zeros(n, np.int32) if shared else np.arange(n, dtype=np.int32)
        yield k, fam, tol, opts, W.Workload(f"options[{k}]", s, q, rho, mid, z, tol), explicit_ids


@pytest.mark.parametrize("seed", [250103330, 250103331])
def test_options_sizes_families(seed):
    import torch
    import paper_2501_03322_b200 as P
    f = lambda a: torch.tensor(a, dtype=torch.float64, device="cuda")
    n_conv = n_beyond = 0
    seen_stage3 = seen_cap = seen_first_only = 0
    for k, fam, tol, opts, wl, explicit_ids in _trials(seed, 40):
        what = (seed, k, fam, tol, opts, wl.n_sources, explicit_ids)
        ctx = P.Context(max(wl.n_sources, 8), **opts)
        r = ctx.twk_magnify(f(wl.s), f(wl.q), f(wl.rho), f(wl.zeta),
                            torch.tensor(wl.model_id, device="cuda") if explicit_ids else None, tol)
        g = {key: v.cpu().numpy() for key, v in r.items()}
        st = g["status"].astype(np.uint32)
        seen_stage3 += ctx.twk_last_stats()["n_stage3"]
        ctx.close()
        o = api.magnify(wl, tol, mode=0, max_samples=opts["max_samples"], subtract_avg_tol=opts["subtract_avg_tol"])
        ref = api.magnify(wl, 1e-7, mode=1)
        fin = np.isfinite(g["mu"])
        assert np.array_equal(fin, np.isfinite(o["mu"])), what
        assert np.all(g["nsamples"][fin] <= opts["max_samples"]) and np.all(g["nsamples"][fin] >= 64), what
        assert np.all(((st[fin] & 1) != 0) ^ ((st[fin] & 2) != 0)), what
        first = fin & (g["nsamples"] == 64) & (o["nsamples"] == 64)
        seen_first_only += int(first.sum())
        if first.any():
            assert np.abs(g["mu"][first] / o["mu"][first] - 1).max() < 1e-7, what
            assert np.array_equal(st[first] & 3, o["status"][first] & 3), what
        rel = np.abs(g["mu"] / ref["mu"] - 1)
        conv = fin & ((st & 1) != 0)
        if conv.any():
            assert rel[conv].max() <= 1.5 * tol, (what, rel[conv].max())
            n_conv += int(conv.sum())
            n_beyond += int((rel[conv] > tol).sum())
        cap = fin & ((st & 2) != 0)
        seen_cap += int(cap.sum())
        if cap.any():
            assert np.all(g["err"][cap] > tol), what
    assert n_beyond <= 2e-3 * n_conv, (n_beyond, n_conv)
    # the trials reached every stage and both exits
    assert seen_stage3 > 0 and seen_cap > 0 and seen_first_only > 0 and n_conv > 1000
