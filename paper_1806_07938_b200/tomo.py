"""ctypes binding of libtomo_b200 (include/tomo.h, include/tomo_host.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of the shared library; PyTorch is used for device buffers
and streams.  There is no CPU fallback: without the built library `load()` raises, and without a CUDA device the
compute calls fail with TOMO_ECUDA.
"""
from __future__ import annotations

import ctypes as C
import math
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtomo_b200.so")

TOMO_OK, TOMO_EINVAL, TOMO_EUNSUPPORTED, TOMO_ENOTREADY, TOMO_ENOMEM, TOMO_ECUDA = 0, -1, -2, -3, -4, -5
TOMO_HUDGIN, TOMO_FRIED, TOMO_FFTMODEL = 0, 1, 2
TOMO_F32, TOMO_F32S_F64A, TOMO_F64 = 0, 1, 2
TOMO_SOLVER_MULTIKERNEL, TOMO_SOLVER_PERSISTENT = 0, 1
TOMO_STATIC_SCRATCH_BYTES = 4194304

EXPORTS = (
    "tomo_plan_create", "tomo_plan_upload_kernels", "tomo_solve", "tomo_solve_batch", "tomo_solve_minres", "tomo_apply_css", "tomo_apply_css_static",
    "tomo_apply_cos", "tomo_cg_step", "tomo_get_zeta", "tomo_time_kernels", "tomo_time_phases", "tomo_time_solver", "tomo_measure_device",
    "tomo_get_sizes", "tomo_get_valid_index", "tomo_get_noise",
    "tomo_get_residuals", "tomo_get_stats", "tomo_get_solver", "tomo_plan_destroy", "tomo_last_error",
    "tomo_host_sizes", "tomo_host_css_generators", "tomo_host_cos_generators", "tomo_host_layer_generators",
    "tomo_host_generator_spectrum",
    "tomo_host_structure_function", "tomo_host_slab_segments",
    "tomo_host_lo_estimator", "tomo_lo_create", "tomo_lo_apply", "tomo_lo_destroy",
)


class TomoError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libtomo_b200 error {code}: {msg}")
        self.code = code


class _Wfs(C.Structure):
    _fields_ = [("ax", C.c_double), ("ay", C.c_double), ("h_gs", C.c_double), ("n_remove", C.c_int)]


class _Geometry(C.Structure):
    _fields_ = [("D", C.c_double), ("n", C.c_int), ("obstruction", C.c_double),
                ("subap_mask", C.POINTER(C.c_ubyte)), ("n_wfs", C.c_int), ("wfs", C.POINTER(_Wfs)),
                ("n_lo", C.c_int), ("lo_wfs", C.POINTER(_Wfs)), ("n_targets", C.c_int),
                ("target_xy", C.POINTER(C.c_double))]


class _Cn2(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("h", C.POINTER(C.c_double)), ("frac", C.POINTER(C.c_double))]


class _Noise(C.Structure):
    _fields_ = [("sigma2_wfs", C.POINTER(C.c_double)), ("noise_frac", C.c_double),
                ("sigma2_subap", C.POINTER(C.c_double)), ("sigma_xy_subap", C.POINTER(C.c_double))]


class _Options(C.Structure):
    _fields_ = [("slope_model", C.c_int), ("pad", C.c_int), ("pad_os", C.c_int), ("max_batch", C.c_int),
                ("precision", C.c_int), ("solver", C.c_int), ("build_cos", C.c_int), ("layered", C.c_int),
                ("fov_radius", C.c_double)]


_lib = None


def load(build_if_missing: bool = True):
    """Load the C-ABI library (building it in-tree first if asked and needed)."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing:
        from . import build as _build
        _build.build()
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1806_07938_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, ip, dp, fp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double), C.c_void_p
    lib.tomo_last_error.restype = C.c_char_p
    lib.tomo_plan_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Cn2), C.c_double, C.c_double,
                                     C.POINTER(_Noise), C.POINTER(_Options), C.POINTER(vp)]
    lib.tomo_plan_upload_kernels.argtypes = [vp, dp, dp]
    lib.tomo_solve.argtypes = [vp, fp, fp, C.c_int, vp]
    lib.tomo_solve_batch.argtypes = [vp, fp, fp, C.c_int, C.c_int, fp, vp]
    lib.tomo_solve_minres.argtypes = [vp, fp, fp, C.c_int, C.c_int, fp, vp]
    lib.tomo_apply_css.argtypes = [vp, fp, fp, vp]
    lib.tomo_apply_css_static.argtypes = [vp, fp, fp, vp]
    lib.tomo_apply_cos.argtypes = [vp, fp, fp, vp]
    lib.tomo_cg_step.argtypes = [vp, fp, fp, fp, vp, vp]
    lib.tomo_get_zeta.argtypes = [vp, fp, C.c_int, vp]
    lib.tomo_time_kernels.argtypes = [vp, C.c_int, C.c_int, C.POINTER(C.c_float), vp]
    lib.tomo_time_phases.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float), vp]
    lib.tomo_time_solver.argtypes = [vp, vp, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_float), vp]
    lib.tomo_get_sizes.argtypes = [vp, ip, ip, ip, ip, ip, ip, ip]
    lib.tomo_get_valid_index.argtypes = [vp, ip, ip]
    lib.tomo_get_noise.argtypes = [vp, dp, dp]
    lib.tomo_get_residuals.argtypes = [vp, dp, C.c_int, C.c_int]
    lib.tomo_get_stats.argtypes = [vp, C.POINTER(C.c_longlong), ip]
    lib.tomo_get_solver.argtypes = [vp, ip, C.c_char_p, C.c_int]
    lib.tomo_plan_destroy.argtypes = [vp]
    lib.tomo_plan_destroy.restype = None
    lib.tomo_host_sizes.argtypes = [C.POINTER(_Geometry), C.POINTER(_Cn2), C.c_int, C.c_int, ip, ip, ip, ip, ip, ip]
    lib.tomo_host_css_generators.argtypes = [C.POINTER(_Geometry), C.POINTER(_Cn2), C.c_double, C.c_double, C.c_int, dp]
    lib.tomo_host_cos_generators.argtypes = [C.POINTER(_Geometry), C.POINTER(_Cn2), C.c_double, C.c_double, C.c_int,
                                             C.c_int, dp]
    lib.tomo_host_layer_generators.argtypes = [C.POINTER(_Geometry), C.POINTER(_Cn2), C.c_double, C.c_double, C.c_int,
                                               C.c_double, ip, dp]
    lib.tomo_host_generator_spectrum.argtypes = [dp, C.c_int, C.c_int, C.c_int, dp]
    lib.tomo_host_structure_function.argtypes = [dp, C.c_int, C.c_double, C.c_double, dp]
    lib.tomo_measure_device.argtypes = [C.c_longlong, C.c_int, C.POINTER(C.c_float), vp]
    lib.tomo_host_slab_segments.argtypes = [C.c_int, C.c_int, C.c_int, ip]
    lib.tomo_host_lo_estimator.argtypes = [C.POINTER(_Geometry), C.POINTER(_Cn2), C.c_double, C.c_double, C.c_int,
                                           C.c_double, dp, dp]
    lib.tomo_lo_create.argtypes = [C.POINTER(_Geometry), C.POINTER(_Cn2), C.c_double, C.c_double, C.c_int, C.c_double,
                                   C.POINTER(vp)]
    lib.tomo_lo_apply.argtypes = [vp, fp, fp, C.c_int, vp]
    lib.tomo_lo_destroy.argtypes = [vp]
    lib.tomo_lo_destroy.restype = None
    _lib = lib
    return lib


def _check(rc: int):
    if rc != TOMO_OK:
        raise TomoError(rc, load().tomo_last_error().decode())


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class _Problem:
    """Keeps the numpy arrays behind the ABI structs alive."""

    def __init__(self, cfg, subap_mask: Optional[np.ndarray] = None, no_targets: bool = False):
        self.cfg = cfg
        self.wfs = (_Wfs * len(cfg.wfs))(*[_Wfs(w.ax, w.ay, w.h_gs, w.n_remove) for w in cfg.wfs])
        lo = getattr(cfg, "lo_wfs", ())
        self.lo = (_Wfs * max(len(lo), 1))(*[_Wfs(w.ax, w.ay, w.h_gs, w.n_remove) for w in lo])
        self.targets = np.ascontiguousarray(np.asarray(() if no_targets else cfg.targets, dtype=np.float64).reshape(-1, 2))
        self.h = np.ascontiguousarray(cfg.h, dtype=np.float64)
        self.frac = np.ascontiguousarray(cfg.frac, dtype=np.float64)
        self.mask = None if subap_mask is None else np.ascontiguousarray(subap_mask, dtype=np.uint8)
        self.geom = _Geometry(cfg.D, cfg.n, cfg.obstruction,
                              None if self.mask is None else self.mask.ctypes.data_as(C.POINTER(C.c_ubyte)),
                              len(cfg.wfs), self.wfs, len(lo), self.lo if len(lo) else None,
                              self.targets.shape[0], _dp(self.targets))
        self.cn2 = _Cn2(len(cfg.h), _dp(self.h), _dp(self.frac))


# ------------------------------------------------------------------------------------------------ host-only (row A0)
def host_sizes(cfg, pad: int = 0, pad_os: int = 0):
    lib = load()
    pr = _Problem(cfg)
    v = [C.c_int() for _ in range(6)]
    _check(lib.tomo_host_sizes(pr.geom, pr.cn2, pad, pad_os, *[C.byref(x) for x in v]))
    return dict(zip(("n_vs", "n_vphi", "n_prime", "P", "P_os", "Kp"), [x.value for x in v]))


def host_css_generators(cfg, slope_model: int = TOMO_HUDGIN) -> np.ndarray:
    lib = load()
    pr = _Problem(cfg)
    Cc, L = 2 * len(cfg.wfs), 2 * cfg.n - 1
    out = np.empty((Cc, Cc, L, L), dtype=np.float64)
    _check(lib.tomo_host_css_generators(pr.geom, pr.cn2, cfg.r0, cfg.L0, slope_model, _dp(out)))
    return out


def host_cos_generators(cfg, target: int = 0, slope_model: int = TOMO_HUDGIN) -> np.ndarray:
    lib = load()
    pr = _Problem(cfg)
    sz = host_sizes(cfg)
    Cc, L = 2 * len(cfg.wfs), sz["n_prime"] + cfg.n - 1
    out = np.empty((sz["Kp"], Cc, L, L), dtype=np.float64)
    _check(lib.tomo_host_cos_generators(pr.geom, pr.cn2, cfg.r0, cfg.L0, slope_model, target, _dp(out)))
    return out


def host_layer_generators(cfg, fov_radius: float, slope_model: int = TOMO_HUDGIN):
    """(n_m, xi'[K][C][n_m+n-1][n_m+n-1]) of a layered plan (L199; reading G31)."""
    lib = load()
    pr = _Problem(cfg, no_targets=True)
    nm = C.c_int()
    _check(lib.tomo_host_layer_generators(pr.geom, pr.cn2, cfg.r0, cfg.L0, slope_model, fov_radius, C.byref(nm), None))
    L = nm.value + cfg.n - 1
    out = np.empty((len(cfg.h), 2 * len(cfg.wfs), L, L), dtype=np.float64)
    _check(lib.tomo_host_layer_generators(pr.geom, pr.cn2, cfg.r0, cfg.L0, slope_model, fov_radius, C.byref(nm), _dp(out)))
    return nm.value, out


def host_generator_spectrum(gen: np.ndarray, n_out: int, n_in: int, P: int) -> np.ndarray:
    lib = load()
    g = np.ascontiguousarray(gen, dtype=np.float64)
    out = np.empty((P // 2 + 1, P, 2), dtype=np.float64)
    _check(lib.tomo_host_generator_spectrum(_dp(g), n_out, n_in, P, _dp(out)))
    return out[..., 0] + 1j * out[..., 1]


def host_structure_function(r, r0: float, L0: float) -> np.ndarray:
    lib = load()
    rr = np.ascontiguousarray(r, dtype=np.float64).ravel()
    out = np.empty_like(rr)
    _check(lib.tomo_host_structure_function(_dp(rr), rr.size, r0, L0, _dp(out)))
    return out.reshape(np.shape(r))


def host_lo_estimator(cfg, sigma2_lo: float, slope_model: int = TOMO_HUDGIN, subap_mask=None):
    """(R_lo [2T][2 n_lo], covariance of the aperture-mean slope pairs [2M][2M]) of tomo_host_lo_estimator."""
    lib = load()
    pr = _Problem(cfg, subap_mask)
    n_lo, T = len(cfg.lo_wfs), len(cfg.targets)
    R = np.empty((2 * T, 2 * n_lo), dtype=np.float64)
    Cm = np.empty((2 * (n_lo + T), 2 * (n_lo + T)), dtype=np.float64)
    _check(lib.tomo_host_lo_estimator(pr.geom, pr.cn2, cfg.r0, cfg.L0, slope_model, sigma2_lo, _dp(R), _dp(Cm)))
    return R, Cm


def measure_device(l2_bytes: int = 0, reps: int = 5, stream=None):
    """L2 -> SM read bandwidth [GB/s] and plain fp32 FMA rate [TFLOP/s] of the current device (tomo_measure_device)."""
    lib = load()
    out = (C.c_float * 2)()
    _check(lib.tomo_measure_device(l2_bytes, reps, out, _stream_handle(stream)))
    return {"l2_read_GBps": float(out[0]), "fp32_TFLOPs": float(out[1])}


def host_slab_segments(Ph: int, n_frames: int, n_ctas: int) -> np.ndarray:
    lib = load()
    out = np.zeros((n_ctas, 8), dtype=np.int32)
    _check(lib.tomo_host_slab_segments(Ph, n_frames, n_ctas, out.ctypes.data_as(C.POINTER(C.c_int))))
    return out


# ------------------------------------------------------------------------------------------------ the plan
def _ptr(t) -> int:
    """Device pointer of a contiguous torch CUDA tensor."""
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return t.data_ptr()


def _stream_handle(stream) -> int:
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream


class LowOrder:
    """tomo_lo_create / tomo_lo_apply / tomo_lo_destroy: the split low-order path of cfg.lo_wfs (include/tomo.h)."""

    def __init__(self, cfg, sigma2_lo: float, slope_model: int = TOMO_HUDGIN, subap_mask=None):
        self.lib = load()
        self._pr = _Problem(cfg, subap_mask)
        self.n_lo, self.n_targets = len(cfg.lo_wfs), len(cfg.targets)
        self._h = C.c_void_p()
        _check(self.lib.tomo_lo_create(self._pr.geom, self._pr.cn2, cfg.r0, cfg.L0, slope_model, sigma2_lo,
                                       C.byref(self._h)))

    def apply(self, lo_slopes, wavefront, stream=None):
        """wavefront [n_frames][T][n_vphi] += tilt estimated from lo_slopes [n_frames][n_lo][2]; in place, asynchronous."""
        n_frames = lo_slopes.shape[0] if lo_slopes.dim() == 3 else 1
        if lo_slopes.numel() != n_frames * self.n_lo * 2 or wavefront.numel() % max(n_frames * self.n_targets, 1):
            raise ValueError("lo_slopes must be [n_frames][n_lo][2] and wavefront [n_frames][T][n_vphi]")
        _check(self.lib.tomo_lo_apply(self._h, _ptr(lo_slopes), _ptr(wavefront), n_frames, _stream_handle(stream)))
        return wavefront

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self.lib.tomo_lo_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class TomoPlan:
    """tomo_plan_create + tomo_plan_upload_kernels; methods mirror the C entry points one to one."""

    def __init__(self, cfg, *, noise_frac: Optional[float] = None, sigma2_wfs: Optional[Sequence[float]] = None,
                 sigma2_subap=None, sigma_xy_subap=None, slope_model: int = TOMO_HUDGIN, max_batch: int = 1, precision: int = TOMO_F32,
                 solver: int = TOMO_SOLVER_PERSISTENT, build_cos: bool = True, subap_mask=None,
                 css_gen: Optional[np.ndarray] = None, cos_gen: Optional[np.ndarray] = None, upload: bool = True,
                 layered: bool = False, fov_radius: float = 0.0):
        """layered=True: the plan estimates every layer on its meta-pupil grid (tomo_options.layered, L199); the targets of
        cfg are ignored and the "wavefront" of the solves is [frame][layer][n_prime][n_prime]."""
        self.lib = load()
        self.cfg = cfg
        self.layered = bool(layered)
        self._pr = _Problem(cfg, subap_mask, no_targets=self.layered)
        if sigma2_subap is not None:
            self._s2 = np.ascontiguousarray(sigma2_subap, dtype=np.float64)
            self._sxy = None if sigma_xy_subap is None else np.ascontiguousarray(sigma_xy_subap, dtype=np.float64)
            noise = _Noise(None, 0.0, _dp(self._s2), None if self._sxy is None else _dp(self._sxy))
        elif sigma2_wfs is not None:
            self._s2 = np.ascontiguousarray(sigma2_wfs, dtype=np.float64)
            noise = _Noise(_dp(self._s2), 0.0, None, None)
        else:
            noise = _Noise(None, cfg.noise_frac if noise_frac is None else noise_frac, None, None)
        opt = _Options(slope_model, cfg.pad, 0 if self.layered else cfg.pad_os, max_batch, precision, solver,
                       1 if build_cos else 0, 1 if self.layered else 0, float(fov_radius))
        self._h = C.c_void_p()
        _check(self.lib.tomo_plan_create(self._pr.geom, self._pr.cn2, cfg.r0, cfg.L0, noise, opt, C.byref(self._h)))
        v = [C.c_int() for _ in range(7)]
        _check(self.lib.tomo_get_sizes(self._h, *[C.byref(x) for x in v]))
        (self.n_vs, self.n_vphi, self.slopes_len, self.wavefront_len, self.P, self.P_os, self.n_prime) = [x.value for x in v]
        self.n_targets = len(cfg.h) if self.layered else len(cfg.targets)     # layered: one n_prime^2 grid per layer
        self.n_wfs = len(cfg.wfs)
        self.max_batch = max_batch
        self.has_cos = build_cos and self.n_targets > 0
        if upload:
            self.upload_kernels(css_gen, cos_gen)

    def upload_kernels(self, css_gen=None, cos_gen=None):
        a = None if css_gen is None else np.ascontiguousarray(css_gen, dtype=np.float64)
        b = None if cos_gen is None else np.ascontiguousarray(cos_gen, dtype=np.float64)
        _check(self.lib.tomo_plan_upload_kernels(self._h, None if a is None else _dp(a), None if b is None else _dp(b)))

    # -- compute entry points (device tensors, asynchronous on the stream) --
    def solve(self, slopes, wavefront_out, n_iter: int, stream=None):
        _check(self.lib.tomo_solve(self._h, _ptr(slopes), _ptr(wavefront_out) if wavefront_out is not None else None,
                                   n_iter, _stream_handle(stream)))

    def solve_batch(self, slopes, wavefront_out, n_frames: int, n_iter: int, x0=None, stream=None):
        _check(self.lib.tomo_solve_batch(self._h, _ptr(slopes),
                                         _ptr(wavefront_out) if wavefront_out is not None else None, n_frames, n_iter,
                                         None if x0 is None else _ptr(x0), _stream_handle(stream)))

    def solve_minres(self, slopes, wavefront_out, n_frames: int, n_iter: int, x0=None, stream=None):
        _check(self.lib.tomo_solve_minres(self._h, _ptr(slopes),
                                          _ptr(wavefront_out) if wavefront_out is not None else None, n_frames, n_iter,
                                          None if x0 is None else _ptr(x0), _stream_handle(stream)))

    def apply_css(self, v, out, stream=None):
        _check(self.lib.tomo_apply_css(self._h, _ptr(v), _ptr(out), _stream_handle(stream)))

    def apply_css_static(self, v, out, stream=None):
        """tomo_apply_css_static: the product with its workspace in the library's static device array (no allocation)."""
        _check(self.lib.tomo_apply_css_static(self._h, _ptr(v), _ptr(out), _stream_handle(stream)))

    def apply_cos(self, zeta, wavefront_out, stream=None):
        _check(self.lib.tomo_apply_cos(self._h, _ptr(zeta), _ptr(wavefront_out), _stream_handle(stream)))

    def cg_step(self, x, r, p, rho_alpha_beta, stream=None):
        _check(self.lib.tomo_cg_step(self._h, _ptr(x), _ptr(r), _ptr(p), _ptr(rho_alpha_beta), _stream_handle(stream)))

    def get_zeta(self, zeta_out, n_frames: int = 1, stream=None):
        _check(self.lib.tomo_get_zeta(self._h, _ptr(zeta_out), n_frames, _stream_handle(stream)))

    def time_kernels(self, n_frames: int, n_iter: int, stream=None):
        ms = (C.c_float * 4)()
        _check(self.lib.tomo_time_kernels(self._h, n_frames, n_iter, ms, _stream_handle(stream)))
        return dict(zip(("rows_fwd", "cols", "rows_inv", "update"), [float(v) for v in ms]))

    def time_phases(self, n_frames: int, n_iter: int, stream=None, minres: bool = False):
        us = (C.c_float * 10)()
        _check(self.lib.tomo_time_phases(self._h, n_frames, n_iter, 1 if minres else 0, us, _stream_handle(stream)))
        return dict(zip(("iteration", "rho_beta", "slab_update", "slab_fft_fwd", "slab_mac", "slab_fft_inv", "barrier_b", "alpha_modes",
                         "rows", "barrier_a"),
                        [float(v) for v in us]))

    def time_solver(self, slopes, n_frames: int, n_iter: int, reps: int, stream=None, minres: bool = False) -> float:
        ms = (C.c_float * 1)()
        _check(self.lib.tomo_time_solver(self._h, _ptr(slopes), n_frames, n_iter, reps, 1 if minres else 0, ms, _stream_handle(stream)))
        return float(ms[0])

    # -- getters --
    def valid_index(self):
        s = np.empty(self.n_vs, dtype=np.int32)
        p = np.empty(self.n_vphi, dtype=np.int32)
        _check(self.lib.tomo_get_valid_index(self._h, s.ctypes.data_as(C.POINTER(C.c_int)),
                                             p.ctypes.data_as(C.POINTER(C.c_int))))
        return s, p

    def noise(self):
        s2 = np.empty(self.n_wfs, dtype=np.float64)
        var = C.c_double()
        _check(self.lib.tomo_get_noise(self._h, _dp(s2), C.byref(var)))
        return s2, var.value

    def residuals(self, n_frames: int, n_iter: int) -> np.ndarray:
        out = np.empty((n_frames, n_iter + 1), dtype=np.float64)
        _check(self.lib.tomo_get_residuals(self._h, _dp(out), n_frames, n_iter))
        return out

    def stats(self):
        b = C.c_longlong()
        n = C.c_int()
        _check(self.lib.tomo_get_stats(self._h, C.byref(b), C.byref(n)))
        return dict(device_bytes=b.value, launches_last_solve=n.value)

    def solver_in_use(self):
        """(TOMO_SOLVER_* that runs this plan, reason the persistent solver was not taken or '')."""
        sv = C.c_int()
        note = C.create_string_buffer(512)
        _check(self.lib.tomo_get_solver(self._h, C.byref(sv), note, 512))
        return sv.value, note.value.decode()

    # -- convenience: host buffers in, host buffers out (H2D + solve + D2H on one stream) --
    def solve_host(self, slopes_host, n_iter: int, n_frames: int = 1, stream=None, minres: bool = False):
        """slopes_host: pinned or pageable torch CPU tensor / numpy array [n_frames][C][n_vs] fp32.
        Returns a pinned CPU tensor [n_frames][n_targets][n_vphi]; the caller synchronises the stream."""
        import torch
        if not hasattr(self, "_hb"):
            self._hb = {}
        key = n_frames
        if key not in self._hb:
            self._hb[key] = (torch.empty(n_frames * self.slopes_len, dtype=torch.float32, device="cuda"),
                             torch.empty(n_frames * self.wavefront_len, dtype=torch.float32, device="cuda"),
                             torch.empty(n_frames * self.wavefront_len, dtype=torch.float32).pin_memory())
        d_in, d_out, h_out = self._hb[key]
        src = slopes_host if isinstance(slopes_host, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(slopes_host, dtype=np.float32))
        s = stream if stream is not None else torch.cuda.current_stream()
        with torch.cuda.stream(s):
            d_in.copy_(src.reshape(-1), non_blocking=True)
            (self.solve_minres if minres else self.solve_batch)(d_in, d_out, n_frames, n_iter, stream=s)
            h_out.copy_(d_out, non_blocking=True)
        return h_out.view(n_frames, self.n_targets, self.n_vphi)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self.lib.tomo_plan_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
