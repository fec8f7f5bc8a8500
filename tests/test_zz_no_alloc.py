"""twk_magnify_static (-m gpu; collected last on purpose): the adaptive path for callers that must not allocate.  Its
workspace is a fixed array inside the library instead of a context's cudaMalloc'ed block (include/twk.h).  Checked
against the existing path -- twk_magnify on a context -- on two calls in a row (the second finds the first call's
contents in the shared array), for different batches, and for the limit."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _device_batch(wl):
    import torch
    dev = torch.device("cuda:0")
    f = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(dt).to(dev)
    mid = None if wl.model_id is None else f(wl.model_id, torch.int32)
    return dict(s=f(wl.s, torch.float64), q=f(wl.q, torch.float64), rho=f(wl.rho, torch.float64), zeta=f(wl.zeta, torch.float64),
                model_id=mid)


def _outputs(n):
    import torch
    dev = torch.device("cuda:0")
    # poisoned: whatever the call does not write shows
    return dict(mu=torch.full((n,), float("nan"), dtype=torch.float64, device=dev),
                err=torch.full((n,), float("nan"), dtype=torch.float64, device=dev),
                nsamples=torch.full((n,), -7, dtype=torch.int32, device=dev),
                status=torch.full((n,), -7, dtype=torch.int32, device=dev))


def _static(d, n, tol):
    import torch
    import paper_2501_03322_b200 as P
    o = _outputs(n)
    rc = P.twk_magnify_static(d["s"], d["q"], d["rho"], d["zeta"], o["mu"], model_id=d["model_id"], rel_tol=tol, out_err=o["err"],
                              out_nsamples=o["nsamples"], out_status=o["status"])
    assert rc == 0
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in o.items()}


def _context(d, n, tol, **opts):
    import torch
    import paper_2501_03322_b200 as P
    c = P.Context(n, **opts)
    r = c.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], tol)
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in r.items()}
    c.close()
    return out


def _cases():
    import workloads as W
    full = W.config4()
    zc = full.zeta[:, 0] + 1j * full.zeta[:, 1]
    band = np.where((np.abs(zc.imag) < 0.25) & (np.abs(zc.real) < 0.6))[0]      # the caustic band: most sources refine
    c5 = W.config5()
    return [(full.subset(band[:: max(1, len(band) // 6000)]), 1e-4),            # ~6,000 sources of the resonant map
            (c5.subset(np.arange(0, 3000)), 1e-6),                               # every source refines, some to the last stage
            (W.config2(), 1e-4)]                                                 # a light curve of 10,000 epochs, one model


def test_static_entry_matches_the_context_path_on_calls_in_a_row():
    import paper_2501_03322_b200 as P
    cases = _cases()
    assert all(wl.n_sources <= P.TWK_STATIC_MAX_SOURCES for wl, _ in cases)
    refs, devs = [], []
    for wl, tol in cases:
        d = _device_batch(wl)
        devs.append(d)
        refs.append((_context(d, wl.n_sources, tol, handoff_slots=0), _context(d, wl.n_sources, tol)))
    # two passes over the batches, back to back: every call but the first finds another call's worklists, seed blocks and
    # records in the shared array
    for rnd in range(2):
        for (wl, tol), d, (lean, dflt) in zip(cases, devs, refs):
            got = _static(d, wl.n_sources, tol)
            assert np.all(np.isfinite(got["mu"])) and np.all(got["nsamples"] >= 64)
            # the same kernels on the same lean layout: the same bits
            assert np.array_equal(got["mu"], lean["mu"]), (rnd, wl.name)
            assert np.array_equal(got["nsamples"], lean["nsamples"]) and np.array_equal(got["status"], lean["status"])
            assert np.array_equal(got["err"], lean["err"])
            # ... and the default context (hand-over arena, stage 1.5) within the tolerance both promise
            rel = np.abs(got["mu"] - dflt["mu"]) / np.abs(dflt["mu"])
            assert rel.max() <= tol, (rnd, wl.name, rel.max())
            assert np.median(rel) < 1e-10


def test_static_entry_rejects_batches_beyond_its_scratch():
    import torch
    import paper_2501_03322_b200 as P
    import workloads as W
    n = P.TWK_STATIC_MAX_SOURCES + 1
    wl = W.config5(n=n)
    d = _device_batch(wl)
    o = _outputs(n)
    rc = P.twk_magnify_static(d["s"], d["q"], d["rho"], d["zeta"], o["mu"], model_id=d["model_id"], rel_tol=1e-4)
    torch.cuda.synchronize()
    assert rc == P.TWK_ELIMIT
    assert b"TWK_STATIC_MAX_SOURCES" in P.lib().twk_strerror(rc)
    assert bool(torch.isnan(o["mu"]).all())                 # nothing was launched
    # exactly at the limit it runs; and an empty batch is a no-op
    wl = W.config5(n=P.TWK_STATIC_MAX_SOURCES)
    d = _device_batch(wl)
    got = _static(d, wl.n_sources, 1e-4)
    ref = _context(d, wl.n_sources, 1e-4, handoff_slots=0)
    assert np.array_equal(got["mu"], ref["mu"]) and np.array_equal(got["nsamples"], ref["nsamples"])
    assert P.twk_magnify_static(d["s"], d["q"], d["rho"], d["zeta"][:0], o["mu"], model_id=None, rel_tol=1e-4) == 0


def test_static_entry_does_not_allocate():
    """Device memory in use is the same before and after a warm call (torch's allocator is not involved: the outputs exist
    beforehand), and the array's size is what the header states."""
    import torch
    import paper_2501_03322_b200 as P
    import workloads as W
    wl = W.config5(n=4000)
    d = _device_batch(wl)
    _static(d, wl.n_sources, 1e-6)                          # first call on the device: address look-up
    o = _outputs(wl.n_sources)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        assert P.twk_magnify_static(d["s"], d["q"], d["rho"], d["zeta"], o["mu"], model_id=d["model_id"], rel_tol=1e-6,
                                    out_err=o["err"], out_nsamples=o["nsamples"], out_status=o["status"]) == 0
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
