"""Python face of the FP64 CPU oracle (oracle/woden_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_2005_09316_b200 and shares no code with it; it
takes plain numpy float64 arrays (the seeded generators in paper_2005_09316_b200/inputs.py
produce them for both sides).

Functions mirror the C-ABI of the CUDA library on HOST arrays, with complex128 output and an
optional `vis_index` (flat (t*F + f)*B + b indices) for subset evaluation.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from . import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp, ip, llp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_longlong)
        common = [C.c_int, C.c_int, C.c_int, dp, dp, dp, dp, C.c_int, dp, dp, dp, dp, C.c_double]
        tail = [llp, C.c_longlong, dp, C.c_int]
        L.woden_oracle_points.argtypes = common + tail
        L.woden_oracle_gaussians.argtypes = common + [dp, dp, dp] + tail
        L.woden_oracle_shapelets.argtypes = common + [dp, dp, dp, dp, ip, ip, ip, dp] + tail
        L.woden_oracle_hermite_functions.argtypes = [C.c_int, C.c_double, dp]
        L.woden_oracle_hermite_functions.restype = None
        L.woden_oracle_tolerance_scale.argtypes = [C.c_int, dp, C.c_int, dp, dp, C.c_double, ip, dp, dp, C.c_int]
        L.woden_oracle_uvw.argtypes = [C.c_int, dp, dp, dp, C.c_int, dp, C.c_double, dp, dp, dp]
        L.woden_oracle_uv_basis.argtypes = [C.c_int, dp, dp, C.c_double, dp]
        for f in (L.woden_oracle_points, L.woden_oracle_gaussians, L.woden_oracle_shapelets,
                  L.woden_oracle_tolerance_scale, L.woden_oracle_uvw, L.woden_oracle_uv_basis):
            f.restype = C.c_int
        _lib = L
    return _lib


def _d(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _pd(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _pi(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_int))


def _prep(u_m, v_m, w_m, freqs_hz, vis_index, out, accumulate):
    u, v, w, fr = _d(u_m), _d(v_m), _d(w_m), _d(freqs_hz)
    if u.ndim != 2 or u.shape != v.shape or u.shape != w.shape:
        raise ValueError("u_m, v_m, w_m must be [T, B] arrays of one shape")
    T, B = u.shape
    F = fr.shape[0]
    if vis_index is not None:
        vi = np.ascontiguousarray(vis_index, dtype=np.int64)
        if vi.size and (vi.min() < 0 or vi.max() >= T * F * B):
            raise ValueError("vis_index out of range")
        shape = (vi.size,)
        pvi = vi.ctypes.data_as(C.POINTER(C.c_longlong))
    else:
        vi, pvi, shape = None, None, (T, F, B)
    if out is None:
        if accumulate:
            raise ValueError("accumulate needs an output array")
        out = np.zeros(shape, dtype=np.complex128)
    if out.dtype != np.complex128 or out.shape != shape or not out.flags.c_contiguous:
        raise ValueError("out must be C-contiguous complex128 of shape %r" % (shape,))
    return u, v, w, fr, T, B, F, vi, pvi, out


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with status {rc}")


def predict_points(u_m, v_m, w_m, freqs_hz, l, m, s0_jy, alpha, ref_freq_hz,
                   vis_index=None, out=None, accumulate=False) -> np.ndarray:
    u, v, w, fr, T, B, F, vi, pvi, out = _prep(u_m, v_m, w_m, freqs_hz, vis_index, out, accumulate)
    l, m, s0, al = _d(l), _d(m), _d(s0_jy), _d(alpha)
    rc = lib().woden_oracle_points(B, T, F, _pd(u), _pd(v), _pd(w), _pd(fr), l.size,
                                   _pd(l), _pd(m), _pd(s0), _pd(al), float(ref_freq_hz),
                                   pvi, 0 if vi is None else vi.size,
                                   out.view(np.float64).ctypes.data_as(C.POINTER(C.c_double)),
                                   int(bool(accumulate)))
    _check(rc, "points")
    return out


def predict_gaussians(u_m, v_m, w_m, freqs_hz, l, m, s0_jy, alpha, ref_freq_hz,
                      maj_fwhm_rad, min_fwhm_rad, pa_rad,
                      vis_index=None, out=None, accumulate=False) -> np.ndarray:
    u, v, w, fr, T, B, F, vi, pvi, out = _prep(u_m, v_m, w_m, freqs_hz, vis_index, out, accumulate)
    l, m, s0, al = _d(l), _d(m), _d(s0_jy), _d(alpha)
    mj, mn, pa = _d(maj_fwhm_rad), _d(min_fwhm_rad), _d(pa_rad)
    rc = lib().woden_oracle_gaussians(B, T, F, _pd(u), _pd(v), _pd(w), _pd(fr), l.size,
                                      _pd(l), _pd(m), _pd(s0), _pd(al), float(ref_freq_hz),
                                      _pd(mj), _pd(mn), _pd(pa),
                                      pvi, 0 if vi is None else vi.size,
                                      out.view(np.float64).ctypes.data_as(C.POINTER(C.c_double)),
                                      int(bool(accumulate)))
    _check(rc, "gaussians")
    return out


def predict_shapelets(u_m, v_m, w_m, freqs_hz, l, m, s0_jy, alpha, ref_freq_hz,
                      beta1_rad, beta2_rad, pa_rad, uv_basis, coeff_offset, n1, n2, coeff,
                      vis_index=None, out=None, accumulate=False) -> np.ndarray:
    u, v, w, fr, T, B, F, vi, pvi, out = _prep(u_m, v_m, w_m, freqs_hz, vis_index, out, accumulate)
    l, m, s0, al = _d(l), _d(m), _d(s0_jy), _d(alpha)
    b1, b2, pa = _d(beta1_rad), _d(beta2_rad), _d(pa_rad)
    M = None if uv_basis is None else _d(uv_basis)
    off, a1, a2, cf = _i(coeff_offset), _i(n1), _i(n2), _d(coeff)
    if off.size != l.size + 1:
        raise ValueError("coeff_offset must have n + 1 entries")
    rc = lib().woden_oracle_shapelets(B, T, F, _pd(u), _pd(v), _pd(w), _pd(fr), l.size,
                                      _pd(l), _pd(m), _pd(s0), _pd(al), float(ref_freq_hz),
                                      _pd(b1), _pd(b2), _pd(pa), _pd(M),
                                      _pi(off), _pi(a1), _pi(a2), _pd(cf),
                                      pvi, 0 if vi is None else vi.size,
                                      out.view(np.float64).ctypes.data_as(C.POINTER(C.c_double)),
                                      int(bool(accumulate)))
    _check(rc, "shapelets")
    return out


def hermite_functions(pmax: int, x: float) -> np.ndarray:
    """h_p(x) = H_p(x) exp(-x^2/2)/sqrt(2^p p!), p = 0..pmax (the oracle's own routine)."""
    out = np.zeros(pmax + 1, dtype=np.float64)
    lib().woden_oracle_hermite_functions(int(pmax), float(x), _pd(out))
    return out


def tolerance_scale(freqs_hz, s0_jy, alpha, ref_freq_hz, coeff_offset=None, coeff=None,
                    out=None) -> np.ndarray:
    """[F] values of sum_k |S_k(nu_f)| w_k (w_k = sum_q |coeff_q| for shapelets, reading G12);
    adds into `out` when given."""
    fr, s0, al = _d(freqs_hz), _d(s0_jy), _d(alpha)
    acc = out is not None
    if out is None:
        out = np.zeros(fr.size, dtype=np.float64)
    off = None if coeff_offset is None else _i(coeff_offset)
    cf = None if coeff is None else _d(coeff)
    rc = lib().woden_oracle_tolerance_scale(fr.size, _pd(fr), s0.size, _pd(s0), _pd(al),
                                            float(ref_freq_hz), _pi(off), _pd(cf), _pd(out), int(acc))
    _check(rc, "tolerance_scale")
    return out


def uvw_from_antennas(x_m, y_m, z_m, hour_angle_rad, dec0_rad):
    """[T, B] u, v, w in metres from local equatorial antenna XYZ (pairs p < q, p-major)."""
    X, Y, Z, H = _d(x_m), _d(y_m), _d(z_m), _d(hour_angle_rad)
    n, T = X.size, H.size
    out = [np.zeros((T, n * (n - 1) // 2), dtype=np.float64) for _ in range(3)]
    _check(lib().woden_oracle_uvw(n, _pd(X), _pd(Y), _pd(Z), T, _pd(H), float(dec0_rad),
                                  _pd(out[0]), _pd(out[1]), _pd(out[2])), "uvw")
    return tuple(out)


def shapelet_uv_basis(l, m, dec0_rad) -> np.ndarray:
    """[n, 6] M_j of reading G4."""
    l, m = _d(np.atleast_1d(l)), _d(np.atleast_1d(m))
    out = np.zeros((l.size, 6), dtype=np.float64)
    _check(lib().woden_oracle_uv_basis(l.size, _pd(l), _pd(m), float(dec0_rad), _pd(out)), "uv_basis")
    return out


def predict_workload(wl, vis_index=None) -> np.ndarray:
    """Total V of a generated workload (all three component types, Eq 11 sums all types)."""
    p, g, s = wl.points, wl.gaussians, wl.shapelets
    out = predict_points(wl.u_m, wl.v_m, wl.w_m, wl.freqs_hz, p.l, p.m, p.s0_jy, p.alpha,
                         wl.ref_freq_hz, vis_index=vis_index)
    if g.n:
        predict_gaussians(wl.u_m, wl.v_m, wl.w_m, wl.freqs_hz, g.l, g.m, g.s0_jy, g.alpha,
                          wl.ref_freq_hz, g.maj_fwhm_rad, g.min_fwhm_rad, g.pa_rad,
                          vis_index=vis_index, out=out, accumulate=True)
    if s.n:
        # M_j (reading G4) from the oracle's own routine, not from the generator's arrays: the CUDA side
        # computes its own too (woden_shapelet_uv_basis), so the two sides share only l, m and dec0
        M = s.uv_basis
        if M is not None and "dec0_rad" in wl.meta:
            M = shapelet_uv_basis(s.l, s.m, wl.meta["dec0_rad"])
        predict_shapelets(wl.u_m, wl.v_m, wl.w_m, wl.freqs_hz, s.l, s.m, s.s0_jy, s.alpha,
                          wl.ref_freq_hz, s.beta1_rad, s.beta2_rad, s.pa_rad, M,
                          s.coeff_offset, s.n1, s.n2, s.coeff,
                          vis_index=vis_index, out=out, accumulate=True)
    return out


def workload_tolerance_scale(wl) -> np.ndarray:
    p, g, s = wl.points, wl.gaussians, wl.shapelets
    sc = tolerance_scale(wl.freqs_hz, p.s0_jy, p.alpha, wl.ref_freq_hz)
    if g.n:
        tolerance_scale(wl.freqs_hz, g.s0_jy, g.alpha, wl.ref_freq_hz, out=sc)
    if s.n:
        tolerance_scale(wl.freqs_hz, s.s0_jy, s.alpha, wl.ref_freq_hz, s.coeff_offset, s.coeff, out=sc)
    return sc
