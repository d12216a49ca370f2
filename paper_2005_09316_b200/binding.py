"""ctypes binding of libwoden_b200.so (include/woden_b200.h).  Argument marshalling only: every
step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device memory
and streams (tensor.data_ptr(), torch.cuda.current_stream()).

There is NO CPU fallback: if the shared library is missing this module raises on first use,
and on a machine without a CUDA device `Woden()` raises `WodenError(WODEN_ERR_CUDA)`.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libwoden_b200.so")

WODEN_OK = 0
WODEN_ERR_NULL = -1
WODEN_ERR_DIM = -2
WODEN_ERR_ORDER = -3
WODEN_ERR_CUDA = -4
WODEN_ERR_UNIMPLEMENTED = -5
WODEN_ERR_DATA = -6
WODEN_ERR_STATIC_LIMIT = -7
WODEN_MAX_ORDER = 100
WODEN_STATIC_TRUNCATE_MAX = 16384
WODEN_EQ25_PIXELS = 257
WODEN_PATH_AUTO = 0
WODEN_PATH_GENERAL = 1
WODEN_PATH_NONE = -1
WODEN_PATH_WALKING = 2
WODEN_SHAPELET_AUTO = 0
WODEN_SHAPELET_REGISTER = 1
WODEN_SHAPELET_TENSOR = 2
WODEN_SHAPELET_REGISTER_SPARSE = 3
WODEN_BASIS_RECURRENCE = 0
WODEN_BASIS_LUT = 1
WODEN_FIT_MAX_ORDER = 86
PIPES = {"FFMA": 0, "MUFU": 1, "DFMA": 2, "I2F": 3, "LOP3": 4, "FFMA2": 5, "FFMA_IMM": 6, "F2F": 7,
         "MUFU_EX2": 8, "MUFU_FFMA": 9, "FFMA_3REG": 10, "FFMA2_3REG": 11, "FFMA2_BCAST": 12, "FFMA2_UR": 13, "WALK": 14}

EXPORTS = ["woden_create", "woden_destroy", "woden_strerror", "woden_last_error", "woden_check",
           "woden_set_path", "woden_last_path", "woden_last_shapelet_path", "woden_last_shapelet_bucket", "woden_kernel_launches", "woden_predict_points", "woden_predict_gaussians",
           "woden_predict_shapelets", "woden_simulate_host", "woden_pipe_rate",
           "woden_uvw_from_antennas", "woden_shapelet_uv_basis", "woden_calibrate_gains", "woden_peel", "woden_set_shapelet_path", "woden_shapelet_series", "woden_fit_shapelets", "woden_fit_gram_ms", "woden_shapelet_basis_sums",
           "woden_shapelet_truncation_weights", "woden_truncate_select", "woden_truncate_select_static", "woden_static_last_error"]

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_vp = C.c_void_p


class woden_uvw(C.Structure):
    _fields_ = [("n_baselines", C.c_int), ("n_times", C.c_int), ("n_freqs", C.c_int),
                ("u_m", _vp), ("v_m", _vp), ("w_m", _vp), ("freqs_hz", _dp)]


class woden_points_host(C.Structure):
    _fields_ = [("n", C.c_int), ("l", _dp), ("m", _dp), ("s0_jy", _dp), ("alpha", _dp)]


class woden_gaussians_host(C.Structure):
    _fields_ = [("n", C.c_int), ("l", _dp), ("m", _dp), ("s0_jy", _dp), ("alpha", _dp),
                ("maj_fwhm_rad", _dp), ("min_fwhm_rad", _dp), ("pa_rad", _dp)]


class woden_shapelets_host(C.Structure):
    _fields_ = [("n", C.c_int), ("n_coeff", C.c_int), ("p_max", C.c_int),
                ("l", _dp), ("m", _dp), ("s0_jy", _dp), ("alpha", _dp),
                ("beta1_rad", _dp), ("beta2_rad", _dp), ("pa_rad", _dp), ("uv_basis", _dp),
                ("coeff_offset", _ip), ("n1", _ip), ("n2", _ip), ("coeff", _dp)]


class woden_image_grid(C.Structure):
    _fields_ = [("n_l", C.c_int), ("n_m", C.c_int), ("dl", C.c_double), ("dm", C.c_double),
                ("l_c", C.c_double), ("m_c", C.c_double)]


class woden_restoring_beam(C.Structure):
    _fields_ = [("bmaj_rad", C.c_double), ("bmin_rad", C.c_double), ("bpa_rad", C.c_double), ("half_width", C.c_int)]


class WodenError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str = ""):
        self.status = status
        super().__init__(f"{what}: status {status} ({detail})")


_lib = None


def load() -> C.CDLL:
    """Load libwoden_b200.so; raises (loudly) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2005_09316_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    L.woden_create.argtypes = [C.POINTER(_vp), C.c_int]
    L.woden_destroy.argtypes = [_vp]
    L.woden_strerror.argtypes = [C.c_int]
    L.woden_strerror.restype = C.c_char_p
    L.woden_last_error.argtypes = [_vp]
    L.woden_last_error.restype = C.c_char_p
    L.woden_check.argtypes = [_vp]
    L.woden_set_path.argtypes = [_vp, C.c_int]
    L.woden_last_path.argtypes = [_vp]
    L.woden_last_shapelet_path.argtypes = [_vp]
    L.woden_last_shapelet_bucket.argtypes = [_vp]
    L.woden_set_shapelet_path.argtypes = [_vp, C.c_int]
    L.woden_shapelet_series.argtypes = [_vp, C.c_int, C.c_int, C.c_longlong, _vp, _vp, C.c_double, C.c_double, _vp, _vp]
    common = [_vp, C.POINTER(woden_uvw), C.c_int, _vp, _vp, _vp, _vp, C.c_double]
    tail = [_vp, C.c_int, _vp]
    L.woden_predict_points.argtypes = common + tail
    L.woden_predict_gaussians.argtypes = common + [_vp, _vp, _vp] + tail
    L.woden_predict_shapelets.argtypes = common + [_vp, _vp, _vp, _vp, _vp, C.c_int, C.c_int, _vp, _vp, _vp] + tail
    L.woden_simulate_host.argtypes = [_vp, C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _dp, C.c_double,
                                      C.POINTER(woden_points_host), C.POINTER(woden_gaussians_host),
                                      C.POINTER(woden_shapelets_host), _vp, _vp]
    L.woden_pipe_rate.argtypes = [_vp, C.c_int, C.c_int, _dp, _dp]
    L.woden_fit_gram_ms.argtypes = [_vp, C.POINTER(C.c_float)]
    L.woden_shapelet_basis_sums.argtypes = [_vp, C.POINTER(woden_image_grid), C.c_double, C.c_double, C.c_double, C.c_int,
                                            C.c_double, C.c_double, C.POINTER(woden_restoring_beam), _vp, _vp]
    L.woden_truncate_select.argtypes = [_vp, C.c_int, _vp, C.c_double, _vp, _vp, _vp]
    L.woden_shapelet_truncation_weights.argtypes = [_vp, C.c_int, _dp, _dp, _dp, _dp, _ip, _ip, _ip, _dp, C.c_int,
                                                    C.c_double, _vp, _vp]
    L.woden_truncate_select_static.argtypes = [C.c_int, _vp, C.c_double, _vp, _vp, _vp]
    L.woden_static_last_error.restype = C.c_char_p
    L.woden_static_last_error.argtypes = []
    L.woden_fit_shapelets.argtypes = [_vp, C.POINTER(woden_image_grid), _vp, C.c_double, C.c_double, C.c_double, C.c_int,
                                      C.c_int, _dp, _dp, C.POINTER(woden_restoring_beam), C.c_int, _vp, _vp, _vp, _vp, _vp]
    L.woden_uvw_from_antennas.argtypes = [_vp, C.c_int, _vp, _vp, _vp, C.c_int, _dp, C.c_double, _vp, _vp, _vp, _vp]
    L.woden_shapelet_uv_basis.argtypes = [_vp, C.c_int, _vp, _vp, C.c_double, _vp, _vp]
    L.woden_calibrate_gains.argtypes = [_vp, C.c_int, C.c_longlong, _vp, _vp, C.c_int, _vp, _vp]
    L.woden_peel.argtypes = [_vp, C.c_int, C.c_longlong, _vp, _vp, _vp, _vp, _vp]
    for name in EXPORTS:
        if name == "woden_kernel_launches":
            L.woden_kernel_launches.restype = C.c_ulonglong
            L.woden_kernel_launches.argtypes = []
        elif name not in ("woden_strerror", "woden_last_error", "woden_static_last_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _ptr(t) -> Optional[int]:
    """Device pointer of a torch tensor (None passes NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return t.data_ptr()


def _stream_handle(stream) -> Optional[int]:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream or None


def _hd(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _hdp(a: Optional[np.ndarray]):
    return None if a is None or a.size == 0 else a.ctypes.data_as(_dp)


def _hip(a: Optional[np.ndarray]):
    return None if a is None or a.size == 0 else a.ctypes.data_as(_ip)


class Uvw:
    """woden_uvw: device u_m, v_m, w_m [T, B] float64 tensors + host channel frequencies."""

    def __init__(self, u_m, v_m, w_m, freqs_hz):
        import torch
        for t in (u_m, v_m, w_m):
            if t.dtype != torch.float64 or t.dim() != 2 or t.shape != u_m.shape:
                raise ValueError("u_m, v_m, w_m must be float64 [T, B] tensors of one shape")
        self.tensors = (u_m, v_m, w_m)
        self.freqs = _hd(freqs_hz)
        self.T, self.B = int(u_m.shape[0]), int(u_m.shape[1])
        self.F = int(self.freqs.shape[0])
        self.c = woden_uvw(self.B, self.T, self.F, _ptr(u_m), _ptr(v_m), _ptr(w_m),
                           self.freqs.ctypes.data_as(_dp))

    @property
    def vis_shape(self):
        return (self.T, self.F, self.B)


class Woden:
    """A woden_ctx.  Methods carry the C entry points' names without the prefix."""

    def __init__(self, device: int = 0):
        self._L = load()
        self._ctx = _vp()
        rc = self._L.woden_create(C.byref(self._ctx), int(device))
        if rc != WODEN_OK:
            self._ctx = None
            raise WodenError(rc, "woden_create", self._L.woden_strerror(rc).decode())
        self.device = int(device)

    def close(self):
        if getattr(self, "_ctx", None):
            self._L.woden_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc: int, what: str):
        if rc != WODEN_OK:
            raise WodenError(rc, what, self._L.woden_strerror(rc).decode() + "; "
                             + self._L.woden_last_error(self._ctx).decode())

    def set_path(self, path: int):
        self._ck(self._L.woden_set_path(self._ctx, int(path)), "woden_set_path")

    def last_path(self) -> int:
        return int(self._L.woden_last_path(self._ctx))

    def last_shapelet_path(self):
        """(engine, order bucket) of the last predict_shapelets call: WODEN_SHAPELET_REGISTER / _REGISTER_SPARSE /
        _TENSOR (WODEN_PATH_NONE, -1 when nothing was launched)."""
        return (int(self._L.woden_last_shapelet_path(self._ctx)), int(self._L.woden_last_shapelet_bucket(self._ctx)))

    def set_shapelet_path(self, path: int):
        self._ck(self._L.woden_set_shapelet_path(self._ctx, int(path)), "woden_set_shapelet_path")

    def check(self):
        self._ck(self._L.woden_check(self._ctx), "woden_check")

    def new_vis(self, uvw: Uvw):
        import torch
        return torch.empty(uvw.vis_shape, dtype=torch.complex64, device=uvw.tensors[0].device)

    def predict_points(self, uvw: Uvw, l, m, s0_jy, alpha, ref_freq_hz, vis, accumulate=False, stream=None):
        n = 0 if l is None else int(l.numel())
        rc = self._L.woden_predict_points(self._ctx, C.byref(uvw.c), n, _ptr(l), _ptr(m), _ptr(s0_jy),
                                          _ptr(alpha), float(ref_freq_hz), _ptr(vis), int(bool(accumulate)),
                                          _stream_handle(stream))
        self._ck(rc, "woden_predict_points")
        return vis

    def predict_gaussians(self, uvw: Uvw, l, m, s0_jy, alpha, ref_freq_hz, maj_fwhm_rad, min_fwhm_rad,
                          pa_rad, vis, accumulate=False, stream=None):
        n = 0 if l is None else int(l.numel())
        rc = self._L.woden_predict_gaussians(self._ctx, C.byref(uvw.c), n, _ptr(l), _ptr(m), _ptr(s0_jy),
                                             _ptr(alpha), float(ref_freq_hz), _ptr(maj_fwhm_rad),
                                             _ptr(min_fwhm_rad), _ptr(pa_rad), _ptr(vis),
                                             int(bool(accumulate)), _stream_handle(stream))
        self._ck(rc, "woden_predict_gaussians")
        return vis

    def predict_shapelets(self, uvw: Uvw, l, m, s0_jy, alpha, ref_freq_hz, beta1_rad, beta2_rad, pa_rad,
                          uv_basis, coeff_offset, n_coeff, p_max, n1, n2, coeff, vis, accumulate=False,
                          stream=None):
        n = 0 if l is None else int(l.numel())
        rc = self._L.woden_predict_shapelets(self._ctx, C.byref(uvw.c), n, _ptr(l), _ptr(m), _ptr(s0_jy),
                                             _ptr(alpha), float(ref_freq_hz), _ptr(beta1_rad), _ptr(beta2_rad),
                                             _ptr(pa_rad), _ptr(uv_basis), _ptr(coeff_offset), int(n_coeff),
                                             int(p_max), _ptr(n1), _ptr(n2), _ptr(coeff), _ptr(vis),
                                             int(bool(accumulate)), _stream_handle(stream))
        self._ck(rc, "woden_predict_shapelets")
        return vis

    def simulate_host(self, wl, vis_host: np.ndarray, stream=None) -> np.ndarray:
        """woden_simulate_host on a generated Workload (host numpy arrays in, complex64 out)."""
        if vis_host.dtype != np.complex64 or not vis_host.flags.c_contiguous:
            raise ValueError("vis_host must be C-contiguous complex64")
        keep = []

        def d(a):
            a = _hd(a); keep.append(a); return _hdp(a)

        def i(a):
            a = np.ascontiguousarray(a, dtype=np.int32); keep.append(a); return _hip(a)

        p, g, s = wl.points, wl.gaussians, wl.shapelets
        cp = woden_points_host(p.n, d(p.l), d(p.m), d(p.s0_jy), d(p.alpha))
        cg = woden_gaussians_host(g.n, d(g.l), d(g.m), d(g.s0_jy), d(g.alpha),
                                  d(g.maj_fwhm_rad) if g.n else None, d(g.min_fwhm_rad) if g.n else None,
                                  d(g.pa_rad) if g.n else None)
        if s.n:
            cs = woden_shapelets_host(s.n, int(s.coeff_offset[-1]), int((s.n1 + s.n2).max()),
                                      d(s.l), d(s.m), d(s.s0_jy), d(s.alpha), d(s.beta1_rad), d(s.beta2_rad),
                                      d(s.pa_rad), d(s.uv_basis) if s.uv_basis is not None else None,
                                      i(s.coeff_offset), i(s.n1), i(s.n2), d(s.coeff))
        else:
            cs = woden_shapelets_host(0, 0, 0)
        u, v, w, fr = _hd(wl.u_m), _hd(wl.v_m), _hd(wl.w_m), _hd(wl.freqs_hz)
        rc = self._L.woden_simulate_host(self._ctx, wl.n_baselines, wl.n_times, wl.n_freqs,
                                         _hdp(u), _hdp(v), _hdp(w), _hdp(fr), float(wl.ref_freq_hz),
                                         C.byref(cp), C.byref(cg), C.byref(cs),
                                         vis_host.ctypes.data_as(_vp), _stream_handle(stream))
        self._ck(rc, "woden_simulate_host")
        return vis_host

    def uvw_from_antennas(self, x_m, y_m, z_m, hour_angle_rad, dec0_rad, stream=None):
        """Device [T, B] u, v, w tensors from device antenna XYZ tensors (woden_uvw_from_antennas)."""
        import torch
        ha = _hd(hour_angle_rad)
        n, T = int(x_m.numel()), int(ha.shape[0])
        out = [torch.empty((T, n * (n - 1) // 2), dtype=torch.float64, device=x_m.device) for _ in range(3)]
        rc = self._L.woden_uvw_from_antennas(self._ctx, n, _ptr(x_m), _ptr(y_m), _ptr(z_m), T, _hdp(ha),
                                             float(dec0_rad), _ptr(out[0]), _ptr(out[1]), _ptr(out[2]),
                                             _stream_handle(stream))
        self._ck(rc, "woden_uvw_from_antennas")
        return tuple(out)

    def shapelet_uv_basis(self, l, m, dec0_rad, stream=None):
        """Device [n, 6] M_j tensor (woden_shapelet_uv_basis)."""
        import torch
        n = int(l.numel())
        out = torch.empty((n, 6), dtype=torch.float64, device=l.device)
        rc = self._L.woden_shapelet_uv_basis(self._ctx, n, _ptr(l), _ptr(m), float(dec0_rad), _ptr(out),
                                             _stream_handle(stream))
        self._ck(rc, "woden_shapelet_uv_basis")
        return out

    def calibrate_gains(self, n_antennas: int, vis_data, vis_model, n_iter: int = 10, stream=None):
        """complex128 gains [..., n_antennas] for complex64 [..., B] device tensors (woden_calibrate_gains)."""
        import torch
        nb = n_antennas * (n_antennas - 1) // 2
        if vis_data.shape != vis_model.shape or vis_data.shape[-1] != nb or vis_data.dtype != torch.complex64:
            raise ValueError("vis_data / vis_model must be complex64 [..., n_ant (n_ant - 1) / 2]")
        cells = vis_data.numel() // nb
        gains = torch.empty(tuple(vis_data.shape[:-1]) + (n_antennas,), dtype=torch.complex128, device=vis_data.device)
        rc = self._L.woden_calibrate_gains(self._ctx, int(n_antennas), cells, _ptr(vis_data), _ptr(vis_model),
                                           int(n_iter), _ptr(gains), _stream_handle(stream))
        self._ck(rc, "woden_calibrate_gains")
        return gains

    def peel(self, n_antennas: int, vis_data, vis_model, gains, out=None, stream=None):
        """V - g_i g_j^* I (woden_peel)."""
        import torch
        nb = n_antennas * (n_antennas - 1) // 2
        cells = vis_data.numel() // nb
        if out is None:
            out = torch.empty_like(vis_data)
        rc = self._L.woden_peel(self._ctx, int(n_antennas), cells, _ptr(vis_data), _ptr(vis_model), _ptr(gains),
                                _ptr(out), _stream_handle(stream))
        self._ck(rc, "woden_peel")
        return out

    def shapelet_series(self, method: int, x, coeff, lut_dx: float = 2.0 ** -7, lut_x_max: float = 32.0, out=None,
                        stream=None):
        """sum_p coeff[p] h_p(x) for a float32 device tensor x (woden_shapelet_series)."""
        import torch
        if x.dtype != torch.float32 or coeff.dtype != torch.float32:
            raise ValueError("x and coeff must be float32 device tensors")
        if out is None:
            out = torch.empty_like(x)
        rc = self._L.woden_shapelet_series(self._ctx, int(method), int(coeff.numel()) - 1, int(x.numel()), _ptr(x),
                                           _ptr(coeff), float(lut_dx), float(lut_x_max), _ptr(out),
                                           _stream_handle(stream))
        self._ck(rc, "woden_shapelet_series")
        return out

    def fit_shapelets(self, image, dl, dm, l_c, m_c, l0, m0, pa_rad, p_max, beta1_rad, beta2_rad, beam=None,
                      n_refine=0, want_weights=False, stream=None):
        """woden_fit_shapelets on a float64 device image [n_m, n_l]; beam = (bmaj, bmin, bpa, half_width) or
        None.  Returns device tensors (coeff [n_beta, P], residual [n_beta], weights or None, best int32[1])."""
        import torch
        if image.dtype != torch.float64 or image.dim() != 2:
            raise ValueError("image must be a float64 [n_m, n_l] device tensor")
        b1, b2 = _hd(np.atleast_1d(beta1_rad)), _hd(np.atleast_1d(beta2_rad))
        if b1.shape != b2.shape:
            raise ValueError("beta1_rad and beta2_rad must have one length")
        n_beta, P = int(b1.shape[0]), (p_max + 1) * (p_max + 2) // 2
        grid = woden_image_grid(int(image.shape[1]), int(image.shape[0]), float(dl), float(dm), float(l_c), float(m_c))
        cb = woden_restoring_beam(*[float(x) for x in beam[:3]], int(beam[3])) if beam is not None else None
        coeff = torch.empty((n_beta, P), dtype=torch.float64, device=image.device)
        resid = torch.empty(n_beta, dtype=torch.float64, device=image.device)
        weights = torch.empty_like(coeff) if want_weights else None
        best = torch.empty(1, dtype=torch.int32, device=image.device)
        rc = self._L.woden_fit_shapelets(self._ctx, C.byref(grid), _ptr(image), float(l0), float(m0), float(pa_rad),
                                         int(p_max), n_beta, _hdp(b1), _hdp(b2), C.byref(cb) if cb is not None else None,
                                         int(n_refine), _ptr(coeff), _ptr(resid), _ptr(weights), _ptr(best),
                                         _stream_handle(stream))
        self._ck(rc, "woden_fit_shapelets")
        return coeff, resid, weights, best

    def shapelet_basis_sums(self, n_l, n_m, dl, dm, l_c, m_c, l0, m0, pa_rad, p_max, beta1_rad, beta2_rad, beam=None,
                            device="cuda:0", stream=None):
        """woden_shapelet_basis_sums: device float64 [P] of sum_pixels |G * B_q| (Eq 25 without |C|)."""
        import torch
        grid = woden_image_grid(int(n_l), int(n_m), float(dl), float(dm), float(l_c), float(m_c))
        cb = woden_restoring_beam(*[float(x) for x in beam[:3]], int(beam[3])) if beam is not None else None
        out = torch.empty((p_max + 1) * (p_max + 2) // 2, dtype=torch.float64, device=device)
        rc = self._L.woden_shapelet_basis_sums(self._ctx, C.byref(grid), float(l0), float(m0), float(pa_rad), int(p_max),
                                               float(beta1_rad), float(beta2_rad), C.byref(cb) if cb is not None else None,
                                               _ptr(out), _stream_handle(stream))
        self._ck(rc, "woden_shapelet_basis_sums")
        return out

    def shapelet_truncation_weights(self, s0_jy, beta1_rad, beta2_rad, pa_rad, coeff_offset, n1, n2, coeff,
                                    n_pix: int = 0, beam_fwhm_rad: float = -1.0, stream=None):
        """woden_shapelet_truncation_weights (Eq 25) on HOST arrays: device float64 [n_coeff] of weights.
        n_pix = 0 / beam_fwhm_rad < 0 take the header's defaults (reading G20)."""
        import torch
        a = [_hd(x) for x in (s0_jy, beta1_rad, beta2_rad, pa_rad)]
        off, i1, i2 = (np.ascontiguousarray(x, dtype=np.int32) for x in (coeff_offset, n1, n2))
        cf = _hd(coeff)
        n = int(a[0].size)
        if off.size != n + 1 or i1.size != cf.size or i2.size != cf.size or (n and int(off[-1]) != cf.size):
            raise ValueError("inconsistent CSR coefficient lists")
        out = torch.empty(int(cf.size), dtype=torch.float64, device=f"cuda:{self.device}")
        ip = lambda x: None if x.size == 0 else x.ctypes.data_as(_ip)
        rc = self._L.woden_shapelet_truncation_weights(self._ctx, n, *[_hdp(x) for x in a], ip(off), ip(i1), ip(i2),
                                                       _hdp(cf), int(n_pix), float(beam_fwhm_rad),
                                                       _ptr(out) if cf.size else None, _stream_handle(stream))
        self._ck(rc, "woden_shapelet_truncation_weights")
        return out

    def truncate_select(self, weights, f_comp: float, stream=None):
        """woden_truncate_select on a float64 device tensor: (keep flags int32 [n], N_comp int32 [1])."""
        import torch
        if weights.dtype != torch.float64 or weights.dim() != 1:
            raise ValueError("weights must be a 1-D float64 device tensor")
        n = int(weights.numel())
        keep = torch.empty(n, dtype=torch.int32, device=weights.device)
        n_keep = torch.empty(1, dtype=torch.int32, device=weights.device)
        rc = self._L.woden_truncate_select(self._ctx, n, _ptr(weights) if n else None, float(f_comp),
                                           _ptr(keep) if n else None, _ptr(n_keep), _stream_handle(stream))
        self._ck(rc, "woden_truncate_select")
        return keep, n_keep

    def fit_gram_ms(self) -> float:
        ms = C.c_float(0.0)
        self._ck(self._L.woden_fit_gram_ms(self._ctx, C.byref(ms)), "woden_fit_gram_ms")
        return float(ms.value)

    def pipe_rate(self, which: str, iters: int = 20000):
        ops, clk = C.c_double(0.0), C.c_double(0.0)
        rc = self._L.woden_pipe_rate(self._ctx, PIPES[which], int(iters), C.byref(ops), C.byref(clk))
        self._ck(rc, "woden_pipe_rate")
        return ops.value, clk.value


def truncate_select_static(weights, f_comp: float, keep, n_keep, stream=None) -> None:
    """woden_truncate_select_static: Eq 23-24 for callers that may not allocate device memory (code
    running inside a framework's fixed device arena, under a memory quota, or in a loop that cannot
    afford cudaMalloc's device-wide stall).  Nothing is allocated here either: `weights` (float64 [n]),
    `keep` (int32 [n]) and `n_keep` (int32 [1]) are the caller's own tensors on the current device, and no
    context is needed.  n above WODEN_STATIC_TRUNCATE_MAX raises WodenError(WODEN_ERR_STATIC_LIMIT).
    Calls share one built-in scratch array per GPU: do not let two of them overlap on the device."""
    import torch
    if weights.dtype != torch.float64 or weights.dim() != 1:
        raise ValueError("weights must be a 1-D float64 device tensor")
    n = int(weights.numel())
    if keep.dtype != torch.int32 or n_keep.dtype != torch.int32 or keep.numel() < n or n_keep.numel() < 1:
        raise ValueError("keep must be int32 [n] and n_keep int32 [1]")
    L = load()
    rc = L.woden_truncate_select_static(n, _ptr(weights) if n else None, float(f_comp), _ptr(keep) if n else None,
                                        _ptr(n_keep), _stream_handle(stream))
    if rc != WODEN_OK:
        raise WodenError(rc, "woden_truncate_select_static: " + L.woden_static_last_error().decode())


def kernel_launches() -> int:
    """Kernels launched by the library since it was loaded (woden_kernel_launches)."""
    return int(load().woden_kernel_launches())


class DeviceWorkload:
    """A generated Workload copied to the GPU once (device-resident inputs for the C-ABI calls).
    With `ctx`, the shapelets' M_j (reading G4) are computed by the library itself
    (woden_shapelet_uv_basis from l, m and the phase-centre declination in wl.meta) instead of being
    copied from the generator's arrays."""

    def __init__(self, wl, device="cuda:0", ctx=None):
        import torch

        def t(a, dtype=torch.float64):
            return None if a is None else torch.as_tensor(np.ascontiguousarray(a), dtype=dtype, device=device)

        self.wl = wl
        self.uvw = Uvw(t(wl.u_m), t(wl.v_m), t(wl.w_m), wl.freqs_hz)
        self.ref = wl.ref_freq_hz
        p, g, s = wl.points, wl.gaussians, wl.shapelets
        self.p = (t(p.l), t(p.m), t(p.s0_jy), t(p.alpha)) if p.n else None
        self.g = (t(g.l), t(g.m), t(g.s0_jy), t(g.alpha), t(g.maj_fwhm_rad), t(g.min_fwhm_rad),
                  t(g.pa_rad)) if g.n else None
        if s.n:
            M = t(s.uv_basis)
            if ctx is not None and s.uv_basis is not None and "dec0_rad" in wl.meta:
                M = ctx.shapelet_uv_basis(t(s.l), t(s.m), wl.meta["dec0_rad"])
            self.s = (t(s.l), t(s.m), t(s.s0_jy), t(s.alpha), t(s.beta1_rad), t(s.beta2_rad), t(s.pa_rad),
                      M, t(s.coeff_offset, torch.int32), int(s.coeff_offset[-1]),
                      int((s.n1 + s.n2).max()), t(s.n1, torch.int32), t(s.n2, torch.int32), t(s.coeff))
        else:
            self.s = None

    def predict(self, ctx: Woden, vis=None, stream=None):
        """The whole hot path in the order shapelets, points, Gaussians (the order woden_simulate_host uses: the
        longest walking call comes last and hides the copy-back); the first non-empty component type overwrites
        `vis`, the others accumulate."""
        if vis is None:
            vis = ctx.new_vis(self.uvw)
        written = False
        if self.s is not None:
            l, m, s0, al, b1, b2, pa, M, off, nc, pmax, n1, n2, cf = self.s
            ctx.predict_shapelets(self.uvw, l, m, s0, al, self.ref, b1, b2, pa, M, off, nc, pmax, n1, n2, cf,
                                  vis, False, stream)
            written = True
        if self.p is not None:
            ctx.predict_points(self.uvw, *self.p, self.ref, vis, written, stream)
            written = True
        if self.g is not None:
            l, m, s0, al, mj, mn, pa = self.g
            ctx.predict_gaussians(self.uvw, l, m, s0, al, self.ref, mj, mn, pa, vis, written, stream)
            written = True
        if not written:         # no components at all: the library zero-fills on an empty overwrite call
            ctx.predict_points(self.uvw, None, None, None, None, self.ref, vis, False, stream)
        return vis
