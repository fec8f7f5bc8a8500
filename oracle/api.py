"""ctypes binding of oracle/libtwk_oracle.so -- TEST INFRASTRUCTURE ONLY.

prec=0 runs the oracle in double (the method's precision), prec=1 in long double (extended twin).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None
_D = C.POINTER(C.c_double)
_I32 = C.POINTER(C.c_int32)
_U32 = C.POINTER(C.c_uint32)
_I8 = C.POINTER(C.c_int8)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_num_threads.restype = C.c_int
        L.orc_coeffs.argtypes = [C.c_double] * 4 + [C.c_int, C.c_int, _D]
        L.orc_quintic_roots.argtypes = [_D, C.c_int, _D]
        L.orc_point.argtypes = [C.c_double] * 6 + [C.c_int, _D, _D, _D, _I32, _D, _D, _I32]
        L.orc_images_fixed.argtypes = [C.c_int64, _D, _D, _D, C.c_int64, _I32, _D, C.c_int, C.c_int, C.c_int,
                                       _D, _I8, _I8, _D, _D, _I32, _D]
        L.orc_magnify.argtypes = [C.c_int64, _D, _D, _D, C.c_int64, _I32, _D, C.c_double, C.c_int, C.c_int, C.c_int,
                                  C.c_int, C.c_int, C.c_int, C.c_int, _D, _D, _I32, _U32, C.c_double, C.c_double, C.c_int]
        L.orc_point_source.argtypes = [C.c_int64, _D, _D, _D, C.c_int64, _I32, _D, C.c_double, C.c_int, _I8, _D, _D, _D]
        L.orc_magnify_thetas.argtypes = [C.c_double] * 6 + [C.c_int] * 5 + [_D]
        L.orc_magnify_thetas.restype = C.c_int
        L.orc_pieces_at.argtypes = [C.c_double] * 5 + [C.c_int, _D, C.c_int, _D, _D, _I32, _I32]
        L.orc_eval_interval_synth.argtypes = [_I32, _D, _D, _D, _I32, _D, _D, _D, C.c_double, _D]
        L.orc_eval_interval_synth.restype = C.c_int
        L.orc_sampler_step.argtypes = [C.c_int, _D, _D, C.c_double, C.c_int, C.c_int, _D]
        L.orc_sampler_step.restype = C.c_int
        L.orc_rayshoot.argtypes = [C.c_double] * 9 + [C.c_int] * 4
        L.orc_rayshoot.restype = C.c_double
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a, t):
    return a.ctypes.data_as(t) if a is not None else None


def _c2(a):
    """float64[..., 2] -> complex128[...]"""
    return a[..., 0] + 1j * a[..., 1]


def coeffs(s, q, zeta, form=6, prec=0):
    """Eq.(6) (form=6) or Eq.(4) (form=4) coefficients c0..c5 (complex128[6]) for CM-frame source position zeta."""
    out = np.zeros(12)
    lib().orc_coeffs(s, q, complex(zeta).real, complex(zeta).imag, form, prec, _p(out, _D))
    return out[0::2] + 1j * out[1::2]


def quintic_roots(c, prec=0):
    cin = np.zeros(12)
    c = np.asarray(c, dtype=np.complex128)
    cin[0::2], cin[1::2] = c.real, c.imag
    out = np.zeros(10)
    lib().orc_quintic_roots(_p(cin, _D), prec, _p(out, _D))
    return out[0::2] + 1j * out[1::2]


def point(s, q, rho, zeta_c, theta, prec=0):
    """One boundary point source.  Returns dict(z, R, J, kind, zp, w, nreal, repaired, sweeps)."""
    z, Res, zp = np.zeros(10), np.zeros(10), np.zeros(10)
    J, w = np.zeros(5), np.zeros(5)
    kind, info = np.zeros(5, np.int32), np.zeros(3, np.int32)
    lib().orc_point(s, q, rho, complex(zeta_c).real, complex(zeta_c).imag, theta, prec, _p(z, _D), _p(Res, _D), _p(J, _D),
                    _p(kind, _I32), _p(zp, _D), _p(w, _D), _p(info, _I32))
    return dict(z=z[0::2] + 1j * z[1::2], R=Res[0::2] + 1j * Res[1::2], J=J, kind=kind, zp=zp[0::2] + 1j * zp[1::2], w=w,
                nreal=int(info[0]), repaired=int(info[1]), sweeps=int(info[2]))


def _batch(wl):
    s = np.ascontiguousarray(wl.s, dtype=np.float64)
    q = np.ascontiguousarray(wl.q, dtype=np.float64)
    rho = np.ascontiguousarray(wl.rho, dtype=np.float64)
    mid = np.ascontiguousarray(wl.model_id, dtype=np.int32)
    zeta = np.ascontiguousarray(wl.zeta, dtype=np.float64)
    return s, q, rho, mid, zeta


def images_fixed(wl, N=None, prec=0, nthreads=0, want_z=True, want_piece=False):
    """Fixed-sampling face over a Workload.  Returns dict(z[n,N,5] complex, kind[n,N,5], count[n,N], mu[n], err[n],
    ncross[n], piece[n,N,2])."""
    N = int(N or wl.fixed_n)
    s, q, rho, mid, zeta = _batch(wl)
    n = zeta.shape[0]
    z = np.zeros((n, N, 5, 2)) if want_z else None
    kind = np.zeros((n, N, 5), np.int8)
    count = np.zeros((n, N), np.int8)
    mu, err = np.zeros(n), np.zeros(n)
    ncross = np.zeros(n, np.int32)
    piece = np.zeros((n, N, 2)) if want_piece else None
    lib().orc_images_fixed(len(s), _p(s, _D), _p(q, _D), _p(rho, _D), n, _p(mid, _I32), _p(zeta, _D), N, prec, nthreads,
                           _p(z, _D), _p(kind, _I8), _p(count, _I8), _p(mu, _D), _p(err, _D), _p(ncross, _I32), _p(piece, _D))
    return dict(z=_c2(z) if want_z else None, kind=kind, count=count, mu=mu, err=err, ncross=ncross, piece=piece)


def magnify(wl, rel_tol=None, mode=0, prec=0, nthreads=0, samples_per_iter=64, initial_samples=64, max_samples=4096,
            subtract_avg_tol=1, slope_gate=1e-5, slope_cos=0.70710678118654752, hidden_guard=0):
    """Adaptive face over a Workload.  mode 0 = the paper's sampler, mode 1 = converged reference (bisection).
    slope_gate: proximity gate of the slope detector (0 = off).  hidden_guard=1 adds the L-4 hidden-crossing
    term to the interval estimates (an extension).  Returns dict(mu, err, nsamples, status)."""
    s, q, rho, mid, zeta = _batch(wl)
    n = zeta.shape[0]
    tol = float(wl.rel_tol if rel_tol is None else rel_tol)
    mu, err = np.zeros(n), np.zeros(n)
    ns = np.zeros(n, np.int32)
    st = np.zeros(n, np.uint32)
    lib().orc_magnify(len(s), _p(s, _D), _p(q, _D), _p(rho, _D), n, _p(mid, _I32), _p(zeta, _D), tol, mode, samples_per_iter,
                      initial_samples, max_samples, subtract_avg_tol, prec, nthreads, _p(mu, _D), _p(err, _D), _p(ns, _I32),
                      _p(st, _U32), float(slope_gate), float(slope_cos), int(hidden_guard))
    return dict(mu=mu, err=err, nsamples=ns, status=st)


def point_source(wl, rel_tol=None, prec=0):
    """N1: point-source adequacy tests over a Workload.  Returns dict(accept bool[n], mu = point source +
    quadrupole term, qrel = relative size of the quadrupole term, A = point-source magnification)."""
    s, q, rho, mid, zeta = _batch(wl)
    n = zeta.shape[0]
    tol = float(wl.rel_tol if rel_tol is None else rel_tol)
    acc = np.zeros(n, np.int8)
    mu, qrel, A = np.zeros(n), np.zeros(n), np.zeros(n)
    lib().orc_point_source(len(s), _p(s, _D), _p(q, _D), _p(rho, _D), n, _p(mid, _I32), _p(zeta, _D), tol, prec, _p(acc, _I8),
                           _p(mu, _D), _p(qrel, _D), _p(A, _D))
    return dict(accept=acc.astype(bool), mu=mu, qrel=qrel, A=A)


def magnify_thetas(s, q, rho, zeta_c, rel_tol, prec=0, samples_per_iter=64, initial_samples=64, max_samples=4096,
                   subtract_avg_tol=1):
    out = np.zeros(max_samples)
    n = lib().orc_magnify_thetas(s, q, rho, complex(zeta_c).real, complex(zeta_c).imag, rel_tol, samples_per_iter,
                                 initial_samples, max_samples, subtract_avg_tol, prec, _p(out, _D))
    return out[:n]


def rayshoot(s, q, rho, zeta_c, box, nx, ny, sub=16, nthreads=0):
    x0, x1, y0, y1 = box
    return float(lib().orc_rayshoot(s, q, rho, complex(zeta_c).real, complex(zeta_c).imag, x0, x1, y0, y1, nx, ny, sub, nthreads))


TERMS = ("E1", "E2", "E3", "E4", "cE1", "cE2", "cE3", "corr")


def pieces_at(s, q, rho, zeta_c, theta, prec=0):
    """Diagnostics: the contour over the sorted angles `theta`.  Returns dict(dA[n], err[n], terms[n,8] (see TERMS),
    cross[n], count[n]); interval i is (theta_i, theta_{i+1}), the last one closes the loop."""
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    n = len(theta)
    piece, terms = np.zeros((n, 2)), np.zeros((n, 8))
    cross, count = np.zeros(n, np.int32), np.zeros(n, np.int32)
    lib().orc_pieces_at(s, q, rho, complex(zeta_c).real, complex(zeta_c).imag, n, _p(theta, _D), prec, _p(piece, _D),
                        _p(terms, _D), _p(cross, _I32), _p(count, _I32))
    return dict(dA=piece[:, 0], err=piece[:, 1], terms=terms, cross=cross, count=count)


def eval_interval_synth(A, B, dth):
    """Diagnostics: eval_interval on two synthetic samples.  A, B = dict(kind int[5], z complex[5], zp complex[5], w float[5]).
    Returns dict(dA, err, terms[8], crossing)."""
    def pack(S):
        z = np.asarray(S["z"], dtype=np.complex128)
        zp = np.asarray(S["zp"], dtype=np.complex128)
        return (np.ascontiguousarray(S["kind"], dtype=np.int32), np.ascontiguousarray(np.stack([z.real, z.imag], 1).ravel()),
                np.ascontiguousarray(np.stack([zp.real, zp.imag], 1).ravel()), np.ascontiguousarray(S["w"], dtype=np.float64))
    ka, za, pa, wa = pack(A)
    kb, zb, pb, wb = pack(B)
    out = np.zeros(10)
    c = lib().orc_eval_interval_synth(_p(ka, _I32), _p(za, _D), _p(pa, _D), _p(wa, _D), _p(kb, _I32), _p(zb, _D), _p(pb, _D),
                                      _p(wb, _D), float(dth), _p(out, _D))
    return dict(dA=out[0], err=out[1], terms=out[2:].copy(), crossing=int(c))


def sampler_step(theta, err, tolA, K=64, subtract_avg_tol=1):
    """Diagnostics: one step of the paper-style sampler on caller-given interval errors.  Returns the new angles."""
    theta = np.ascontiguousarray(theta, dtype=np.float64)
    err = np.ascontiguousarray(err, dtype=np.float64)
    out = np.zeros(K)
    m = lib().orc_sampler_step(len(theta), _p(theta, _D), _p(err, _D), float(tolA), int(K), int(subtract_avg_tol), _p(out, _D))
    return out[:m]
