"""ctypes binding of libtwk.so (include/twk.h).  Same names as the C entry points; marshalling only.

Device buffers are torch CUDA tensors (PyTorch is used for device memory and streams, nothing else); their
data_ptr() goes straight into the C ABI.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
# TWK_LIBRARY selects another build of the same sources (the -DTWK_DEBUG build libtwk_debug.so of tests/test_gpu_debug.py)
_LIB_PATH = os.environ.get("TWK_LIBRARY") or os.path.join(HERE, "libtwk.so")
_lib = None

TWK_ST_CONVERGED, TWK_ST_CAP, TWK_ST_REPAIRED, TWK_ST_DOMAIN, TWK_ST_NUMERIC, TWK_ST_SLOPE, TWK_ST_POINT = 1, 2, 4, 8, 16, 32, 64

SYMBOLS = ["twk_default_options", "twk_create", "twk_destroy", "twk_workspace_bytes", "twk_magnify", "twk_magnify_lightcurve", "twk_magnify_lightcurve_orbital",
           "twk_images_fixed", "twk_images_fixed_seeded", "twk_stage1_records",
           "twk_coeffs_eq6", "twk_magnify_host", "twk_magnify_static", "twk_last_stats", "twk_enable_stage_timing", "twk_last_stage_ms", "twk_fp64_peak_probe", "twk_debug_counters", "twk_strerror", "twk_version"]


class TwkError(RuntimeError):
    pass


class twk_options(C.Structure):
    _fields_ = [("max_samples", C.c_int),
                ("subtract_avg_tol", C.c_int), ("handoff_slots", C.c_int64), ("slope_gate", C.c_double), ("slope_cos", C.c_double), ("point_source_test", C.c_int), ("hidden_crossing_guard", C.c_int), ("frame", C.c_int)]


def library_path() -> str:
    return _LIB_PATH


def lib():
    """Load libtwk.so; fails loudly when it has not been built (python -m paper_2501_03322_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise TwkError(f"{_LIB_PATH} is missing: build it with __graft_entry__.build() "
                           "(nvcc, sm_100a); there is no CPU fallback")
        L = C.CDLL(_LIB_PATH)
        vp, sz, dbl, i32 = C.c_void_p, C.c_size_t, C.c_double, C.c_int
        L.twk_default_options.argtypes = [C.POINTER(twk_options)]
        L.twk_default_options.restype = None
        L.twk_create.argtypes = [C.POINTER(vp), C.POINTER(twk_options), sz]
        L.twk_destroy.argtypes = [vp]
        L.twk_workspace_bytes.argtypes = [C.POINTER(twk_options), sz]
        L.twk_workspace_bytes.restype = sz
        L.twk_magnify.argtypes = [vp, sz, vp, vp, vp, sz, vp, vp, dbl, vp, vp, vp, vp, vp]
        L.twk_magnify_lightcurve.argtypes = [vp, sz, vp, vp, vp, vp, vp, vp, vp, sz, vp, vp, dbl, vp, vp, vp, vp, vp]
        L.twk_magnify_lightcurve_orbital.argtypes = [vp, sz, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp, vp, dbl, vp, vp, vp, vp, vp]
        L.twk_magnify_host.argtypes = [vp, sz, vp, vp, vp, sz, vp, vp, dbl, vp, vp, vp, vp, vp]
        L.twk_magnify_static.argtypes = [sz, vp, vp, vp, sz, vp, vp, dbl, vp, vp, vp, vp, vp]
        L.twk_images_fixed.argtypes = [vp, sz, vp, vp, vp, sz, vp, vp, i32, vp, vp, vp, vp, vp, vp]
        L.twk_images_fixed_seeded.argtypes = [vp, sz, vp, vp, vp, sz, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp]
        L.twk_stage1_records.argtypes = [vp, sz, vp, vp, vp, sz, vp, vp, vp, vp, vp]
        L.twk_coeffs_eq6.argtypes = [vp, sz, vp, vp, sz, vp, vp, vp, vp]
        L.twk_last_stats.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int), vp]
        L.twk_enable_stage_timing.argtypes = [vp, i32]
        L.twk_last_stage_ms.argtypes = [vp, C.POINTER(C.c_float)]
        L.twk_fp64_peak_probe.argtypes = [i32, C.POINTER(dbl)]
        L.twk_debug_counters.argtypes = [C.POINTER(C.c_uint32), i32]
        L.twk_strerror.argtypes = [i32]
        L.twk_strerror.restype = C.c_char_p
        L.twk_version.restype = C.c_char_p
        _lib = L
    return _lib


def exported_symbols():
    """Names include/twk.h declares that the loaded library exports (used by the CPU-side ABI test)."""
    L = lib()
    return [s for s in SYMBOLS if hasattr(L, s)]


def _check(rc: int, what: str):
    if rc != 0:
        raise TwkError(f"{what} failed: {lib().twk_strerror(rc).decode()} ({rc})")


def _options(**kw) -> twk_options:
    o = twk_options()
    lib().twk_default_options(C.byref(o))
    for k, v in kw.items():
        if not hasattr(o, k):
            raise TypeError(f"unknown option {k}")
        setattr(o, k, float(v) if k in ("slope_gate", "slope_cos") else int(v))
    return o


def twk_workspace_bytes(max_sources: int, **opts) -> int:
    return int(lib().twk_workspace_bytes(C.byref(_options(**opts)), max_sources))


def twk_version() -> str:
    return lib().twk_version().decode()


def twk_debug_counters(reset: bool = False):
    """Invariant-violation counters of the debug build (raises TwkError on the release build)."""
    out = (C.c_uint32 * 12)()
    _check(lib().twk_debug_counters(out, 1 if reset else 0), "twk_debug_counters")
    return [int(x) for x in out]


TWK_STATIC_MAX_SOURCES = 16384   # include/twk.h
TWK_ELIMIT = -4


def twk_magnify_static(s, q, rho, zeta, out_mu, model_id=None, rel_tol=1e-4, out_err=None, out_nsamples=None, out_status=None,
                       stream=None):
    """twk_magnify without a context and without any allocation: the workspace is a fixed array inside the library
    (include/twk.h).  All tensors CUDA and caller-owned, outputs included (this wrapper allocates nothing either);
    at most TWK_STATIC_MAX_SOURCES sources; calls on one device must not overlap.  Returns the library's code
    (0, or TWK_ELIMIT for a batch beyond the limit); other errors raise."""
    n = int(zeta.shape[0])
    rc = lib().twk_magnify_static(int(s.shape[0]), _ptr(s), _ptr(q), _ptr(rho), n, _ptr(model_id), _ptr(zeta), float(rel_tol),
                                  _ptr(out_mu), _ptr(out_err), _ptr(out_nsamples), _ptr(out_status), _stream_ptr(stream))
    if rc != TWK_ELIMIT:
        _check(rc, "twk_magnify_static")
    return rc


def twk_fp64_peak_probe(iters: int = 1 << 16) -> float:
    out = C.c_double()
    _check(lib().twk_fp64_peak_probe(iters, C.byref(out)), "twk_fp64_peak_probe")
    return out.value


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr(stream=None):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


class Context:
    """twk_ctx wrapper: owns the device workspace for up to max_sources sources per call."""

    def __init__(self, max_sources: int, **opts):
        import torch
        if not torch.cuda.is_available():
            raise TwkError("no CUDA device: the twk hot path has no CPU fallback")
        self._h = C.c_void_p()
        self.max_sources = int(max_sources)
        self.options = _options(**opts)
        _check(lib().twk_create(C.byref(self._h), C.byref(self.options), self.max_sources), "twk_create")

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().twk_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:      # interpreter shutdown: module globals may already be gone
            pass

    # -- device-pointer calls -----------------------------------------------------------------------------------
    def twk_magnify(self, s, q, rho, zeta, model_id=None, rel_tol=1e-4, out_mu=None, out_err=None, out_nsamples=None,
                    out_status=None, want=("err", "nsamples", "status"), stream=None):
        """s, q, rho: float64 CUDA tensors [n_models]; zeta: float64 CUDA [n_sources, 2]; model_id: int32 CUDA or None.
        Returns dict(mu, err, nsamples, status) of CUDA tensors (asynchronous on the stream)."""
        import torch
        n = int(zeta.shape[0])
        dev = zeta.device
        for t_, dt in ((s, torch.float64), (q, torch.float64), (rho, torch.float64), (zeta, torch.float64)):
            assert t_.is_cuda and t_.dtype == dt and t_.is_contiguous()
        if model_id is not None:
            assert model_id.is_cuda and model_id.dtype == torch.int32 and model_id.is_contiguous()
        if out_mu is None:
            out_mu = torch.empty(n, dtype=torch.float64, device=dev)
        if out_err is None and "err" in want:
            out_err = torch.empty(n, dtype=torch.float64, device=dev)
        if out_nsamples is None and "nsamples" in want:
            out_nsamples = torch.empty(n, dtype=torch.int32, device=dev)
        if out_status is None and "status" in want:
            out_status = torch.empty(n, dtype=torch.int32, device=dev)     # uint32 bit patterns
        _check(lib().twk_magnify(self._h, int(s.shape[0]), _ptr(s), _ptr(q), _ptr(rho), n, _ptr(model_id), _ptr(zeta),
                                 float(rel_tol), _ptr(out_mu), _ptr(out_err), _ptr(out_nsamples), _ptr(out_status),
                                 _stream_ptr(stream)), "twk_magnify")
        return dict(mu=out_mu, err=out_err, nsamples=out_nsamples, status=out_status)

    def twk_magnify_lightcurve(self, s, q, rho, t0, u0, tE, alpha, t, model_id=None, rel_tol=1e-4, stream=None):
        """Light-curve front end: per-model trajectory parameters (float64 CUDA [n_models]) and per-source epochs t
        (float64 CUDA [n_sources]); the source centres are computed on the device.  Returns dict like twk_magnify."""
        import torch
        n = int(t.shape[0])
        dev = t.device
        mu = torch.empty(n, dtype=torch.float64, device=dev)
        err = torch.empty(n, dtype=torch.float64, device=dev)
        ns = torch.empty(n, dtype=torch.int32, device=dev)
        st = torch.empty(n, dtype=torch.int32, device=dev)
        _check(lib().twk_magnify_lightcurve(self._h, int(s.shape[0]), _ptr(s), _ptr(q), _ptr(rho), _ptr(t0), _ptr(u0), _ptr(tE),
                                            _ptr(alpha), n, _ptr(model_id), _ptr(t), float(rel_tol), _ptr(mu), _ptr(err),
                                            _ptr(ns), _ptr(st), _stream_ptr(stream)), "twk_magnify_lightcurve")
        return dict(mu=mu, err=err, nsamples=ns, status=st)

    def twk_magnify_lightcurve_orbital(self, s, q, rho, t0, u0, tE, alpha, ds_dt, dalpha_dt, t, model_id=None, rel_tol=1e-4,
                                       stream=None):
        """Light-curve front end with first-order lens orbital motion: as twk_magnify_lightcurve plus the per-model rates
        ds_dt, dalpha_dt (float64 CUDA [n_models]); every epoch gets its own lens on the device."""
        import torch
        n = int(t.shape[0])
        dev = t.device
        mu = torch.empty(n, dtype=torch.float64, device=dev)
        err = torch.empty(n, dtype=torch.float64, device=dev)
        ns = torch.empty(n, dtype=torch.int32, device=dev)
        st = torch.empty(n, dtype=torch.int32, device=dev)
        _check(lib().twk_magnify_lightcurve_orbital(self._h, int(s.shape[0]), _ptr(s), _ptr(q), _ptr(rho), _ptr(t0), _ptr(u0),
                                                    _ptr(tE), _ptr(alpha), _ptr(ds_dt), _ptr(dalpha_dt), n, _ptr(model_id),
                                                    _ptr(t), float(rel_tol), _ptr(mu), _ptr(err), _ptr(ns), _ptr(st),
                                                    _stream_ptr(stream)), "twk_magnify_lightcurve_orbital")
        return dict(mu=mu, err=err, nsamples=ns, status=st)

    def twk_images_fixed(self, s, q, rho, zeta, N, model_id=None, want_z=True, want_kind=True, stream=None):
        import torch
        n = int(zeta.shape[0])
        dev = zeta.device
        z = torch.empty((n, N, 5, 2), dtype=torch.float64, device=dev) if want_z else None
        kind = torch.empty((n, N, 5), dtype=torch.int8, device=dev) if want_kind else None
        count = torch.empty((n, N), dtype=torch.int8, device=dev)
        mu = torch.empty(n, dtype=torch.float64, device=dev)
        err = torch.empty(n, dtype=torch.float64, device=dev)
        _check(lib().twk_images_fixed(self._h, int(s.shape[0]), _ptr(s), _ptr(q), _ptr(rho), n, _ptr(model_id), _ptr(zeta),
                                      int(N), _ptr(z), _ptr(kind), _ptr(count), _ptr(mu), _ptr(err), _stream_ptr(stream)),
               "twk_images_fixed")
        return dict(z=z, kind=kind, count=count, mu=mu, err=err)

    def twk_images_fixed_seeded(self, s, q, rho, zeta, N, model_id=None, stream=None):
        """As twk_images_fixed with the adaptive kernels' solver; adds diag = uint32[4] {solves, recoveries, cold, guard}."""
        import torch
        n = int(zeta.shape[0])
        dev = zeta.device
        z = torch.empty((n, N, 5, 2), dtype=torch.float64, device=dev)
        kind = torch.empty((n, N, 5), dtype=torch.int8, device=dev)
        count = torch.empty((n, N), dtype=torch.int8, device=dev)
        mu = torch.empty(n, dtype=torch.float64, device=dev)
        err = torch.empty(n, dtype=torch.float64, device=dev)
        diag = torch.zeros(4, dtype=torch.int32, device=dev)
        _check(lib().twk_images_fixed_seeded(self._h, int(s.shape[0]), _ptr(s), _ptr(q), _ptr(rho), n, _ptr(model_id),
                                             _ptr(zeta), int(N), _ptr(z), _ptr(kind), _ptr(count), _ptr(mu), _ptr(err),
                                             _ptr(diag), _stream_ptr(stream)), "twk_images_fixed_seeded")
        return dict(z=z, kind=kind, count=count, mu=mu, err=err, diag=diag)

    def twk_stage1_records(self, s, q, rho, zeta, model_id=None, stream=None):
        """The first-iteration records of the stage-1 kernel: dict(records float64[n, 26, 64], diag int32[4])."""
        import torch
        n = int(zeta.shape[0])
        dev = zeta.device
        rec = torch.zeros((n, 26, 64), dtype=torch.float64, device=dev)
        diag = torch.zeros(4, dtype=torch.int32, device=dev)
        _check(lib().twk_stage1_records(self._h, int(s.shape[0]), _ptr(s), _ptr(q), _ptr(rho), n, _ptr(model_id), _ptr(zeta),
                                        _ptr(rec), _ptr(diag), _stream_ptr(stream)), "twk_stage1_records")
        return dict(records=rec, diag=diag)

    def twk_coeffs_eq6(self, s, q, zeta, model_id=None, stream=None):
        """Eq.(6) coefficients of the point source at every zeta as the device builder computes them: complex128[n, 6]."""
        import torch
        n = int(zeta.shape[0])
        out = torch.zeros((n, 6, 2), dtype=torch.float64, device=zeta.device)
        _check(lib().twk_coeffs_eq6(self._h, int(s.shape[0]), _ptr(s), _ptr(q), n, _ptr(model_id), _ptr(zeta), _ptr(out),
                                    _stream_ptr(stream)), "twk_coeffs_eq6")
        o = out.cpu().numpy()
        return o[..., 0] + 1j * o[..., 1]

    # -- host-buffer call (end to end) -----------------------------------------------------------------------------
    def twk_magnify_host(self, s, q, rho, zeta, model_id=None, rel_tol=1e-4, out=None, stream=None):
        """Host buffers: numpy arrays or (pinned) CPU torch tensors, float64 / int32, C-contiguous.  Synchronous.
        `out` may hold preallocated host outputs dict(mu, err, nsamples, status)."""
        def hp(a):
            if a is None:
                return None
            if isinstance(a, np.ndarray):
                assert a.flags.c_contiguous
                return C.c_void_p(a.ctypes.data)
            return C.c_void_p(a.data_ptr())
        n = int(zeta.shape[0])
        if out is None:
            out = dict(mu=np.empty(n), err=np.empty(n), nsamples=np.empty(n, np.int32), status=np.empty(n, np.uint32))
        _check(lib().twk_magnify_host(self._h, int(s.shape[0]), hp(s), hp(q), hp(rho), n, hp(model_id), hp(zeta),
                                      float(rel_tol), hp(out["mu"]), hp(out.get("err")), hp(out.get("nsamples")),
                                      hp(out.get("status")), _stream_ptr(stream)), "twk_magnify_host")
        return out

    def twk_last_stats(self, stream=None):
        a, b, c = C.c_int64(), C.c_int64(), C.c_int()
        _check(lib().twk_last_stats(self._h, C.byref(a), C.byref(b), C.byref(c), _stream_ptr(stream)), "twk_last_stats")
        return dict(n_stage2=a.value, n_stage3=b.value, n_launches=c.value)

    def twk_enable_stage_timing(self, on=True):
        _check(lib().twk_enable_stage_timing(self._h, 1 if on else 0), "twk_enable_stage_timing")

    def twk_last_stage_ms(self):
        ms = (C.c_float * 4)()
        _check(lib().twk_last_stage_ms(self._h, ms), "twk_last_stage_ms")
        return dict(stage0=ms[0], stage1=ms[1], stage2=ms[2], stage3=ms[3])

    # -- convenience over a workloads.Workload ------------------------------------------------------------------------
    def upload(self, wl, device="cuda"):
        import torch
        t = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(device=device, dtype=dt)
        return dict(s=t(wl.s, torch.float64), q=t(wl.q, torch.float64), rho=t(wl.rho, torch.float64),
                    zeta=t(wl.zeta, torch.float64), model_id=t(wl.model_id, torch.int32))

    def magnify_workload(self, wl, rel_tol=None):
        d = self.upload(wl)
        r = self.twk_magnify(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"], wl.rel_tol if rel_tol is None else rel_tol)
        return {k: v.cpu().numpy() for k, v in r.items()}

    def images_fixed_workload(self, wl, N=None, seeded=False):
        d = self.upload(wl)
        f = self.twk_images_fixed_seeded if seeded else self.twk_images_fixed
        r = f(d["s"], d["q"], d["rho"], d["zeta"], int(N or wl.fixed_n), d["model_id"])
        o = {k: v.cpu().numpy() for k, v in r.items()}
        o["z"] = o["z"][..., 0] + 1j * o["z"][..., 1]
        return o

    def stage1_records_workload(self, wl):
        """Stage-1 records unpacked like images_fixed_workload (N = 64): z complex[n, 64, 5], kind int8[n, 64, 5] (by record
        slot: a 3-image sample holds its ghosts in slots 1 and 4), count int8[n, 64], flags int[n, 64], diag."""
        d = self.upload(wl)
        r = self.twk_stage1_records(d["s"], d["q"], d["rho"], d["zeta"], d["model_id"])
        rec = r["records"].cpu().numpy()                                  # [n, 26, 64]
        z = np.moveaxis(rec[:, 0:5, :] + 1j * rec[:, 5:10, :], 1, 2)      # [n, 64, 5]
        code = np.ascontiguousarray(rec[:, 25, :]).view(np.int64)
        count = (code & 7).astype(np.int8)
        kind = np.empty(z.shape, np.int8)
        kind[...] = np.array([1, 1, -1, -1, -1], np.int8)
        three = count == 3
        kind[three, 1] = 0
        kind[three, 4] = 0
        return dict(z=z, kind=kind, count=count, flags=(code >> 3).astype(np.int32), diag=r["diag"].cpu().numpy(),
                    zp=np.moveaxis(rec[:, 10:15, :] + 1j * rec[:, 15:20, :], 1, 2), w=np.moveaxis(rec[:, 20:25, :], 1, 2))
