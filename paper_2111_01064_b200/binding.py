"""Thin ctypes binding over libll_b200.so — same names as include/ll.h, argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory
(`tensor.data_ptr()`) and the current stream.  There is no CPU fallback: if the shared library is missing
or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "libll_b200.so")

LL_OK, LL_ERR_ARG, LL_ERR_STATE, LL_ERR_CUDA, LL_ERR_NOMEM, LL_ERR_UNSUPPORTED, LL_ERR_REF_ZERO = 0, -1, -2, -3, -4, -5, -6
LL_PREC_FP64, LL_PREC_FP32_ACC = 0, 1
LL_STATIC_SCRATCH_BYTES = 2 * 1024 * 1024  # include/ll.h: the static device array of ll_pt_stretch_half_het_static
LL_BC_NATURAL, LL_BC_NOT_A_KNOT = 0, 1

# every symbol include/ll.h declares (tests/test_abi.py checks header and library against this list)
SYMBOLS = (
    "ll_create", "ll_destroy", "ll_last_error", "ll_abi_version", "ll_debug_check", "ll_set_data", "ll_get_dd", "ll_standin_config",
    "ll_standin_split_tc",
    "ll_full_batch", "ll_full_batch_pw", "ll_full_batch_tf", "ll_tlm_nodes", "ll_standin_nodes", "ll_full_batch_standin", "ll_full_batch_standin_host",
    "ll_full_template_standin",
    "ll_template_standin", "ll_het_prepare", "ll_het_refresh_standin", "ll_het_audit_standin",
    "ll_pt_stretch_half_het", "ll_pt_stretch_half_het_static", "ll_pt_stretch_half_full", "ll_pt_swap", "ll_pt_stats", "ll_pt_run_het", "ll_pt_run_full", "ll_pt_fused", "ll_stop_snr", "ll_stop_converged", "ll_het_get_summary", "ll_het_batch", "ll_het_batch_standin",
    "ll_het_batch_standin_host", "ll_peak_fma", "ll_kernel_launches", "ll_last_full_stats",
    "ll_profile_enable", "ll_profile_read",
)


class LLError(RuntimeError):
    def __init__(self, code: int, what: str, text: str = ""):
        super().__init__(f"{what} failed with status {code}" + (f": {text}" if text else ""))
        self.code = code


class ll_config(C.Structure):
    _fields_ = [("device", C.c_int32), ("n_channels", C.c_int32), ("n_modes", C.c_int32), ("precision", C.c_int32),
                ("spline_bc", C.c_int32), ("reserved", C.c_int32 * 3)]


_lib = None


def load_library(path: Optional[str] = None):
    """dlopen libll_b200.so (built by `paper_2111_01064_b200.build`); fails loudly if it is absent."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or SO_PATH
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not found: run `python -m paper_2111_01064_b200.build` "
                                "(the CUDA extension is required; there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, i64, i32, dbl = C.c_void_p, C.c_int64, C.c_int32, C.c_double
    sig = {
        "ll_create": (C.c_int, [C.POINTER(ll_config), C.POINTER(vp)]),
        "ll_destroy": (C.c_int, [vp]),
        "ll_last_error": (C.c_char_p, [vp]),
        "ll_abi_version": (C.c_int, []),
        "ll_debug_check": (C.c_int, [vp, C.POINTER(i32)]),
        "ll_set_data": (C.c_int, [vp, i64, i64, dbl, vp, vp, i32, vp]),
        "ll_standin_split_tc": (C.c_int, [vp, i32]),
        "ll_get_dd": (C.c_int, [vp, C.POINTER(dbl), C.POINTER(dbl), vp]),
        "ll_standin_config": (C.c_int, [vp, i32, vp, vp, vp, dbl]),
        "ll_full_batch": (C.c_int, [vp, i64, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]),
        "ll_full_batch_tf": (C.c_int, [vp, i64, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]),
        "ll_full_batch_pw": (C.c_int, [vp, i64, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]),
        "ll_tlm_nodes": (C.c_int, [vp, i64, i32, vp, vp, dbl, vp, vp]),
        "ll_standin_nodes": (C.c_int, [vp, i64, i32, vp, vp, vp, vp, vp, vp]),
        "ll_full_batch_standin": (C.c_int, [vp, i64, i32, vp, vp, vp, vp, vp, vp]),
        "ll_full_batch_standin_host": (C.c_int, [vp, i64, i32, vp, vp, vp, vp, vp, vp]),
        "ll_full_template_standin": (C.c_int, [vp, i32, vp, vp, vp, vp]),
        "ll_template_standin": (C.c_int, [vp, vp, i64, vp, dbl, dbl, vp, vp]),
        "ll_het_prepare": (C.c_int, [vp, i32, vp, vp, vp, vp]),
        "ll_het_get_summary": (C.c_int, [vp, vp, vp, vp, vp, vp]),
        "ll_het_batch": (C.c_int, [vp, i64, vp, vp, vp, vp, vp, vp, vp, vp]),
        "ll_het_batch_standin": (C.c_int, [vp, i64, vp, vp, vp, vp, vp]),
        "ll_het_refresh_standin": (C.c_int, [vp, i64, vp, vp, i32, vp, vp, vp]),
        "ll_het_audit_standin": (C.c_int, [vp, i64, vp, vp, vp, vp, vp]),
        "ll_pt_stretch_half_het": (C.c_int, [vp, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, i32, dbl, vp, vp, vp, vp, vp]),
        "ll_pt_stretch_half_het_static": (C.c_int, [vp, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, i32, dbl, vp, vp, vp, vp, vp]),
        "ll_pt_stretch_half_full": (C.c_int, [vp, i32, vp, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, i32, dbl, vp, vp, vp,
                                              vp, vp]),
        "ll_pt_swap": (C.c_int, [vp, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp]),
        "ll_pt_run_het": (C.c_int, [vp, i32, i32, vp, vp, vp, vp, vp, vp, vp, i32, dbl, C.c_uint64, i64, i64, vp, vp]),
        "ll_pt_run_full": (C.c_int, [vp, i32, vp, i32, i32, vp, vp, vp, vp, vp, vp, vp, i32, dbl, C.c_uint64, i64, i64, vp,
                                     vp]),
        "ll_pt_stats": (C.c_int, [vp, i64, vp, vp, vp, vp, vp]),
        "ll_pt_fused": (C.c_int, [vp, i32]),
        "ll_stop_snr": (C.c_int, [dbl, dbl]),
        "ll_stop_converged": (C.c_int, [vp, dbl]),
        "ll_het_batch_standin_host": (C.c_int, [vp, i64, vp, vp, vp, vp, vp]),
        "ll_peak_fma": (C.c_int, [vp, i32, i64, C.POINTER(dbl), C.POINTER(dbl), vp]),
        "ll_kernel_launches": (i64, [vp]),
        "ll_last_full_stats": (C.c_int, [vp, C.POINTER(dbl), C.POINTER(i64), vp]),
        "ll_profile_enable": (C.c_int, [vp, i32]),
        "ll_profile_read": (C.c_int, [vp, C.POINTER(dbl), C.POINTER(i64)]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    if path == SO_PATH:
        _lib = lib
    return lib


def _torch():
    import torch
    return torch


def _dev_ptr_i32(t, what: str):
    """device pointer of a contiguous int32 CUDA tensor (None -> NULL)"""
    if t is None:
        return None
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.int32 and t.is_contiguous()):
        raise TypeError(f"{what}: need a contiguous int32 CUDA tensor")
    return C.c_void_p(t.data_ptr())


def _dev_ptr(t, what: str):
    """device pointer of a contiguous float64 CUDA tensor (None -> NULL)"""
    if t is None:
        return None
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{what}: need a contiguous float64 CUDA tensor")
    return C.c_void_p(t.data_ptr())


def _shape(t, shape, what: str):
    """marshalling guard: a wrong shape would read or write out of bounds on the device (None passes)"""
    if t is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{what}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return t


def _host_f64(a, what: str) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.ndim < 1:
        raise TypeError(f"{what}: need an array")
    return a


def _stream_ptr(stream=None, device=None):
    torch = _torch()
    s = torch.cuda.current_stream(device) if stream is None else stream
    return C.c_void_p(s.cuda_stream)


class StopState(C.Structure):
    """ll_stop_state (include/ll.h): Module-2 stopping function state"""
    _fields_ = [("n_checks", C.c_int32), ("count", C.c_int32), ("has_ref", C.c_int32), ("reserved", C.c_int32),
                ("tol", C.c_double), ("ref", C.c_double)]


def stop_snr(extracted_snr: float, limit: float) -> bool:
    return bool(load_library().ll_stop_snr(float(extracted_snr), float(limit)))


def stop_converged(state: StopState, max_logL: float) -> bool:
    return bool(load_library().ll_stop_converged(C.byref(state), float(max_logL)))


class Context:
    """One `ll_ctx` (include/ll.h).  Methods carry the C names without the `ll_` prefix."""

    def __init__(self, n_modes: int = 1, precision: int = LL_PREC_FP64, device: Optional[int] = None, n_channels: int = 2,
                 spline_bc: int = 0):
        torch = _torch()
        if not torch.cuda.is_available():
            raise LLError(LL_ERR_CUDA, "ll_create", "no CUDA device (there is no CPU fallback)")
        self._lib = load_library()
        self.device = torch.cuda.current_device() if device is None else int(device)
        self.n_modes, self.n_channels, self.precision = int(n_modes), int(n_channels), int(precision)
        cfg = ll_config(self.device, self.n_channels, self.n_modes, self.precision, int(spline_bc), (C.c_int32 * 3)(0, 0, 0))
        h = C.c_void_p()
        rc = self._lib.ll_create(C.byref(cfg), C.byref(h))
        if rc != LL_OK:
            raise LLError(rc, "ll_create")
        self._h = h
        self.n_f = 0

    # -- plumbing
    def _check(self, rc: int, what: str):
        if rc != LL_OK:
            raise LLError(rc, what, self.last_error())

    def last_error(self) -> str:
        return (self._lib.ll_last_error(self._h) or b"").decode()

    def debug_check(self) -> int:
        """number of internal buffers whose guard band was written (out-of-bounds stores); 0 = clean"""
        n = C.c_int32(-1)
        self._check(self._lib.ll_debug_check(self._h, C.byref(n)), "ll_debug_check")
        return int(n.value)

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.ll_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    @property
    def P(self) -> int:
        return 5 + 2 * self.n_channels * self.n_modes

    def _out(self, n_w: int, want: bool = True):
        torch = _torch()
        return torch.empty(n_w, dtype=torch.float64, device=f"cuda:{self.device}") if want else None

    # -- F0
    def set_data(self, n_f: int, k_min: int, df: float, d, W, stream=None):
        """d [n_c][n_f][2]; W [n_f] (one weight row for every channel: w_shared = 1) or [n_c][n_f] (w_shared = 0)"""
        n_f = int(n_f)
        w_shared = 1
        if n_f > 0:  # sizes the library cannot see; n_f <= 0 is the library's own argument error
            if d.numel() != self.n_channels * n_f * 2:
                raise ValueError(f"d: expected {self.n_channels} x {n_f} x 2 values, got {tuple(d.shape)}")
            w_shared = 1 if W.numel() == n_f else 0
            if not w_shared:
                _shape(W, (self.n_channels, n_f), "W")
        self._check(self._lib.ll_set_data(self._h, n_f, int(k_min), float(df), _dev_ptr(d, "d"), _dev_ptr(W, "W"), w_shared,
                                          _stream_ptr(stream, self.device)), "ll_set_data")
        self.n_f = n_f

    def get_dd(self, stream=None):
        a, b = C.c_double(), C.c_double()
        self._check(self._lib.ll_get_dd(self._h, C.byref(a), C.byref(b), _stream_ptr(stream, self.device)), "ll_get_dd")
        return a.value, b.value

    def standin_config(self, l, m, c_lm, kappa: float):
        l = np.ascontiguousarray(l, dtype=np.int32)
        m = np.ascontiguousarray(m, dtype=np.int32)
        c = _host_f64(c_lm, "c_lm")
        if not (len(l) == len(m) == len(c)):
            raise ValueError("l, m, c_lm: one entry per mode each")
        self._check(self._lib.ll_standin_config(self._h, len(m), l.ctypes.data_as(C.c_void_p), m.ctypes.data_as(C.c_void_p),
                                                c.ctypes.data_as(C.c_void_p), float(kappa)), "ll_standin_config")

    def standin_split_tc(self, on: bool = True):
        """stand-in full-grid entry points: keep 2 pi f t_c outside the spline as t_shift = t_c (reading R32)"""
        self._check(self._lib.ll_standin_split_tc(self._h, 1 if on else 0), "ll_standin_split_tc")

    def _check_nodes(self, n_w, n_nodes, amp, phase, tf, band, t_shift):
        _shape(amp, (n_w, self.n_modes, n_nodes), "amp")
        _shape(phase, (n_w, self.n_modes, n_nodes), "phase")
        _shape(tf, (n_w, self.n_modes, self.n_channels, 2), "tf")
        _shape(band, (n_w, 2), "band")
        _shape(t_shift, (n_w,), "t_shift")

    # -- full-grid path
    def full_batch(self, f_nodes, amp, phase, tf, band=None, want_parts: bool = True, t_shift=None, stream=None):
        f_nodes = _host_f64(f_nodes, "f_nodes")
        n_w = int(amp.shape[0]) if amp is not None else 0
        self._check_nodes(n_w, len(f_nodes), amp, phase, tf, band, t_shift)
        logL, d_h, h_h = self._out(n_w), self._out(n_w, want_parts), self._out(n_w, want_parts)
        self._check(self._lib.ll_full_batch(self._h, n_w, len(f_nodes), f_nodes.ctypes.data_as(C.c_void_p),
                                            _dev_ptr(amp, "amp"), _dev_ptr(phase, "phase"), _dev_ptr(tf, "tf"),
                                            _dev_ptr(band, "band"), _dev_ptr(t_shift, "t_shift"),
                                            _dev_ptr(logL, "logL"), _dev_ptr(d_h, "d_h"),
                                            _dev_ptr(h_h, "h_h"), _stream_ptr(stream, self.device)), "ll_full_batch")
        return logL, d_h, h_h

    def full_batch_pw(self, f_nodes_w, amp, phase, tf, band=None, want_parts: bool = True, out=None, t_shift=None,
                      stream=None):
        """per-walker node grids: f_nodes_w [n_w][n_nodes] on the device (reading R30)"""
        n_w, n_nodes = int(f_nodes_w.shape[0]), int(f_nodes_w.shape[1])
        self._check_nodes(n_w, n_nodes, amp, phase, tf, band, t_shift)
        logL, d_h, h_h = out if out is not None else (self._out(n_w), self._out(n_w, want_parts), self._out(n_w, want_parts))
        for o in (logL, d_h, h_h):
            _shape(o, (n_w,), "output")
        self._check(self._lib.ll_full_batch_pw(self._h, n_w, n_nodes, _dev_ptr(f_nodes_w, "f_nodes_w"), _dev_ptr(amp, "amp"),
                                               _dev_ptr(phase, "phase"), _dev_ptr(tf, "tf"), _dev_ptr(band, "band"),
                                               _dev_ptr(t_shift, "t_shift"),
                                               _dev_ptr(logL, "logL"), _dev_ptr(d_h, "d_h"), _dev_ptr(h_h, "h_h"),
                                               _stream_ptr(stream, self.device)), "ll_full_batch_pw")
        return logL, d_h, h_h

    def full_batch_tf(self, f_nodes, amp, phase, tf_nodes, band=None, want_parts: bool = True, out=None, t_shift=None,
                      stream=None):
        """frequency-dependent transfer function: tf_nodes [n_w][n_m][n_c][n_nodes][2] (Eq. 8-9)"""
        f_nodes = _host_f64(f_nodes, "f_nodes")
        n_w = int(amp.shape[0]) if amp is not None else 0
        self._check_nodes(n_w, len(f_nodes), amp, phase, None, band, t_shift)
        _shape(tf_nodes, (n_w, self.n_modes, self.n_channels, len(f_nodes), 2), "tf_nodes")
        logL, d_h, h_h = out if out is not None else (self._out(n_w), self._out(n_w, want_parts), self._out(n_w, want_parts))
        for o in (logL, d_h, h_h):
            _shape(o, (n_w,), "output")
        self._check(self._lib.ll_full_batch_tf(self._h, n_w, len(f_nodes), f_nodes.ctypes.data_as(C.c_void_p),
                                               _dev_ptr(amp, "amp"), _dev_ptr(phase, "phase"),
                                               _dev_ptr(tf_nodes, "tf_nodes"), _dev_ptr(band, "band"),
                                               _dev_ptr(t_shift, "t_shift"),
                                               _dev_ptr(logL, "logL"), _dev_ptr(d_h, "d_h"), _dev_ptr(h_h, "h_h"),
                                               _stream_ptr(stream, self.device)), "ll_full_batch_tf")
        return logL, d_h, h_h

    def standin_nodes(self, f_nodes, params, with_band=False, stream=None):
        """stand-in node arrays in the caller layout: amp, phase [n_w][n_m][n_nodes] (radians); with_band: also the
        walkers' bands [n_w][2] (reading R10)"""
        f_nodes = _host_f64(f_nodes, "f_nodes")
        torch = _torch()
        n_w = int(params.shape[0])
        _shape(params, (n_w, self.P), "params")
        amp = torch.empty((n_w, self.n_modes, len(f_nodes)), dtype=torch.float64, device=params.device)
        phase = torch.empty_like(amp)
        band = torch.empty((n_w, 2), dtype=torch.float64, device=params.device) if with_band else None
        self._check(self._lib.ll_standin_nodes(self._h, n_w, len(f_nodes), f_nodes.ctypes.data_as(C.c_void_p),
                                               _dev_ptr(params, "params"), _dev_ptr(amp, "amp"), _dev_ptr(phase, "phase"),
                                               _dev_ptr(band, "band") if with_band else None,
                                               _stream_ptr(stream, self.device)), "ll_standin_nodes")
        return (amp, phase, band) if with_band else (amp, phase)

    def tlm_nodes(self, f_nodes, phase, t_ref: float, stream=None):
        """t_lm(f_j) = t_ref - (1/2pi) dphi/df at the nodes (Eq. 8); phase [n_w][n_m][n_nodes] radians"""
        f_nodes = _host_f64(f_nodes, "f_nodes")
        torch = _torch()
        _shape(phase, (int(phase.shape[0]), self.n_modes, len(f_nodes)), "phase")
        out = torch.empty_like(phase)
        self._check(self._lib.ll_tlm_nodes(self._h, int(phase.shape[0]), len(f_nodes), f_nodes.ctypes.data_as(C.c_void_p),
                                           _dev_ptr(phase, "phase"), float(t_ref), _dev_ptr(out, "t_lm"),
                                           _stream_ptr(stream, self.device)), "ll_tlm_nodes")
        return out

    def _check_rows(self, params, out):
        n_w = int(params.shape[0])
        _shape(params, (n_w, self.P), "params")
        if out is not None:
            for o in out:
                _shape(o, (n_w,), "output")
        return n_w

    def full_batch_standin(self, f_nodes, params, out=None, stream=None):
        f_nodes = _host_f64(f_nodes, "f_nodes")
        n_w = self._check_rows(params, out)
        logL, d_h, h_h = out if out is not None else (self._out(n_w), self._out(n_w), self._out(n_w))
        self._check(self._lib.ll_full_batch_standin(self._h, n_w, len(f_nodes), f_nodes.ctypes.data_as(C.c_void_p),
                                                    _dev_ptr(params, "params"), _dev_ptr(logL, "logL"),
                                                    _dev_ptr(d_h, "d_h"), _dev_ptr(h_h, "h_h"), _stream_ptr(stream, self.device)),
                    "ll_full_batch_standin")
        return logL, d_h, h_h

    def full_batch_standin_host(self, f_nodes, params_host, out_host, stream=None):
        """params_host, out_host = (logL, d_h, h_h): pinned CPU float64 tensors (or numpy arrays)."""
        f_nodes = _host_f64(f_nodes, "f_nodes")
        n_w = self._check_rows(params_host, out_host)
        ptr = lambda t: None if t is None else C.c_void_p(t.data_ptr() if hasattr(t, "data_ptr") else t.ctypes.data)
        self._check(self._lib.ll_full_batch_standin_host(self._h, n_w, len(f_nodes), f_nodes.ctypes.data_as(C.c_void_p),
                                                         ptr(params_host), ptr(out_host[0]), ptr(out_host[1]),
                                                         ptr(out_host[2]), _stream_ptr(stream, self.device)),
                    "ll_full_batch_standin_host")
        return out_host

    def full_template_standin(self, f_nodes, params_row, stream=None):
        torch = _torch()
        f_nodes = _host_f64(f_nodes, "f_nodes")
        row = _host_f64(params_row, "params_row")
        assert row.shape == (self.P,)
        h = torch.empty((self.n_channels, self.n_f, 2), dtype=torch.float64, device=f"cuda:{self.device}")
        self._check(self._lib.ll_full_template_standin(self._h, len(f_nodes), f_nodes.ctypes.data_as(C.c_void_p),
                                                       row.ctypes.data_as(C.c_void_p), _dev_ptr(h, "h"),
                                                       _stream_ptr(stream, self.device)), "ll_full_template_standin")
        return h

    def template_standin(self, params_row, f, f_lo: float, f_hi: float, stream=None):
        torch = _torch()
        row = _host_f64(params_row, "params_row")
        assert row.shape == (self.P,)
        h = torch.empty((self.n_channels, f.shape[0], 2), dtype=torch.float64, device=f"cuda:{self.device}")
        self._check(self._lib.ll_template_standin(self._h, row.ctypes.data_as(C.c_void_p), int(f.shape[0]), _dev_ptr(f, "f"),
                                                  float(f_lo), float(f_hi), _dev_ptr(h, "h"), _stream_ptr(stream, self.device)),
                    "ll_template_standin")
        return h

    # -- heterodyned path
    def het_prepare(self, f_edges, h0_dense, h0_edges, stream=None):
        f_edges = _host_f64(f_edges, "f_edges")
        _shape(h0_dense, (self.n_channels, self.n_f, 2), "h0_dense")
        _shape(h0_edges, (self.n_channels, len(f_edges), 2), "h0_edges")
        self._n_edges = len(f_edges)
        self._check(self._lib.ll_het_prepare(self._h, len(f_edges), f_edges.ctypes.data_as(C.c_void_p),
                                             _dev_ptr(h0_dense, "h0_dense"), _dev_ptr(h0_edges, "h0_edges"),
                                             _stream_ptr(stream, self.device)), "ll_het_prepare")

    def het_get_summary(self, stream=None):
        n_b = self._n_edges - 1
        A0, A1 = np.empty((self.n_channels, n_b, 2)), np.empty((self.n_channels, n_b, 2))
        B0, B1 = np.empty((self.n_channels, n_b)), np.empty((self.n_channels, n_b))
        p = lambda a: a.ctypes.data_as(C.c_void_p)
        self._check(self._lib.ll_het_get_summary(self._h, p(A0), p(A1), p(B0), p(B1), _stream_ptr(stream, self.device)),
                    "ll_het_get_summary")
        return dict(A0=A0, A1=A1, B0=B0, B1=B1)

    def het_batch(self, amp_e, phase_e, tf, t_shift=None, stream=None):
        n_w = int(amp_e.shape[0])
        self._check_nodes(n_w, getattr(self, "_n_edges", int(amp_e.shape[-1])), amp_e, phase_e, tf, None, t_shift)
        logL, d_h, h_h = self._out(n_w), self._out(n_w), self._out(n_w)
        self._check(self._lib.ll_het_batch(self._h, n_w, _dev_ptr(amp_e, "amp_e"), _dev_ptr(phase_e, "phase_e"),
                                           _dev_ptr(tf, "tf"), _dev_ptr(t_shift, "t_shift"),
                                           _dev_ptr(logL, "logL"), _dev_ptr(d_h, "d_h"),
                                           _dev_ptr(h_h, "h_h"), _stream_ptr(stream, self.device)), "ll_het_batch")
        return logL, d_h, h_h

    def het_batch_standin(self, params, out=None, stream=None):
        n_w = self._check_rows(params, out)
        logL, d_h, h_h = out if out is not None else (self._out(n_w), self._out(n_w), self._out(n_w))
        self._check(self._lib.ll_het_batch_standin(self._h, n_w, _dev_ptr(params, "params"), _dev_ptr(logL, "logL"),
                                                   _dev_ptr(d_h, "d_h"), _dev_ptr(h_h, "h_h"), _stream_ptr(stream, self.device)),
                    "ll_het_batch_standin")
        return logL, d_h, h_h

    def het_refresh_standin(self, params, logL, n_edges: int, stream=None):
        """reference update: best walker -> h0 -> summary data; returns (best_index, f_edges)"""
        best = C.c_int64(-1)
        _shape(params, (int(params.shape[0]), self.P), "params")
        _shape(logL, (int(params.shape[0]),), "logL")
        f_edges = np.empty(int(n_edges), dtype=np.float64)
        self._check(self._lib.ll_het_refresh_standin(self._h, int(params.shape[0]), _dev_ptr(params, "params"),
                                                     _dev_ptr(logL, "logL"), int(n_edges), C.byref(best),
                                                     f_edges.ctypes.data_as(C.c_void_p), _stream_ptr(stream, self.device)),
                    "ll_het_refresh_standin")
        self._n_edges = int(n_edges)
        return best.value, f_edges

    def het_audit_standin(self, params, out=None, stream=None):
        """brute-force dense log L over the heterodyne band"""
        n_w = self._check_rows(params, out)
        logL, d_h, h_h = out if out is not None else (self._out(n_w), self._out(n_w), self._out(n_w))
        self._check(self._lib.ll_het_audit_standin(self._h, n_w, _dev_ptr(params, "params"), _dev_ptr(logL, "logL"),
                                                   _dev_ptr(d_h, "d_h"), _dev_ptr(h_h, "h_h"), _stream_ptr(stream, self.device)),
                    "ll_het_audit_standin")
        return logL, d_h, h_h

    # -- sampler step (readings R25-R28): x [n_temps][n_walkers][P], everything on the device
    def pt_stretch_half(self, half, x, logL, d_h, h_h, betas, lo, hi, n_dim, u_z, u_partner, u_accept, a=2.0,
                        accepted=None, f_nodes=None, stream=None):
        """stretch move on one half of every temperature, in place; f_nodes given -> full-grid likelihood, else het"""
        n_t, n_w = int(x.shape[0]), int(x.shape[1])
        self._check_pt(x, logL, d_h, h_h, betas, lo, hi)
        for u in (u_z, u_partner, u_accept):
            _shape(u, (n_t, n_w // 2), "u_z / u_partner / u_accept")
        _shape(accepted, (n_t, n_w // 2), "accepted")
        tail = (n_t, n_w, int(half), _dev_ptr(x, "x"), _dev_ptr(logL, "logL"), _dev_ptr(d_h, "d_h"), _dev_ptr(h_h, "h_h"),
                _dev_ptr(betas, "betas"), _dev_ptr(lo, "lo"), _dev_ptr(hi, "hi"), int(n_dim), float(a), _dev_ptr(u_z, "u_z"),
                _dev_ptr(u_partner, "u_partner"), _dev_ptr(u_accept, "u_accept"), _dev_ptr_i32(accepted, "accepted"),
                _stream_ptr(stream, self.device))
        if f_nodes is None:
            self._check(self._lib.ll_pt_stretch_half_het(self._h, *tail), "ll_pt_stretch_half_het")
        else:
            f_nodes = _host_f64(f_nodes, "f_nodes")
            self._check(self._lib.ll_pt_stretch_half_full(self._h, len(f_nodes), f_nodes.ctypes.data_as(C.c_void_p), *tail),
                        "ll_pt_stretch_half_full")

    def pt_stretch_half_static(self, half, x, logL, d_h, h_h, betas, lo, hi, n_dim, u_z, u_partner, u_accept, a=2.0,
                               accepted=None, stream=None):
        """pt_stretch_half on the heterodyned likelihood with the step's scratch in the library's static device array
        (LL_STATIC_SCRATCH_BYTES, one per GPU, shared by all calls): the call allocates nothing; sizes beyond the array
        raise LLError (include/ll.h: ll_pt_stretch_half_het_static)"""
        n_t, n_w = int(x.shape[0]), int(x.shape[1])
        self._check_pt(x, logL, d_h, h_h, betas, lo, hi)
        for u in (u_z, u_partner, u_accept):
            _shape(u, (n_t, n_w // 2), "u_z / u_partner / u_accept")
        _shape(accepted, (n_t, n_w // 2), "accepted")
        self._check(self._lib.ll_pt_stretch_half_het_static(
            self._h, n_t, n_w, int(half), _dev_ptr(x, "x"), _dev_ptr(logL, "logL"), _dev_ptr(d_h, "d_h"), _dev_ptr(h_h, "h_h"),
            _dev_ptr(betas, "betas"), _dev_ptr(lo, "lo"), _dev_ptr(hi, "hi"), int(n_dim), float(a), _dev_ptr(u_z, "u_z"),
            _dev_ptr(u_partner, "u_partner"), _dev_ptr(u_accept, "u_accept"), _dev_ptr_i32(accepted, "accepted"),
            _stream_ptr(stream, self.device)), "ll_pt_stretch_half_het_static")

    def _check_pt(self, x, logL, d_h, h_h, betas, lo, hi):
        n_t, n_w = int(x.shape[0]), int(x.shape[1])
        _shape(x, (n_t, n_w, self.P), "x")
        for v in (logL, d_h, h_h):
            _shape(v, (n_t, n_w), "logL / d_h / h_h")
        _shape(betas, (n_t,), "betas")
        _shape(lo, (self.P,), "lo")
        _shape(hi, (self.P,), "hi")

    def pt_run(self, x, logL, d_h, h_h, betas, lo, hi, n_dim, seed, iter0, n_iter, a=2.0, n_accepted=None, f_nodes=None,
               stream=None):
        """n_iter whole iterations with the library's counter-based uniforms (reading R31); n_accepted: int64 CUDA
        tensor [n_temps] the accepted proposals are added to, or None"""
        torch = _torch()
        if n_accepted is not None and not (n_accepted.is_cuda and n_accepted.dtype == torch.int64 and n_accepted.is_contiguous()):
            raise TypeError("n_accepted: need a contiguous int64 CUDA tensor")
        acc = None if n_accepted is None else C.c_void_p(n_accepted.data_ptr())
        self._check_pt(x, logL, d_h, h_h, betas, lo, hi)
        _shape(n_accepted, (int(x.shape[0]),), "n_accepted")
        tail = (int(x.shape[0]), int(x.shape[1]), _dev_ptr(x, "x"), _dev_ptr(logL, "logL"), _dev_ptr(d_h, "d_h"),
                _dev_ptr(h_h, "h_h"), _dev_ptr(betas, "betas"), _dev_ptr(lo, "lo"), _dev_ptr(hi, "hi"), int(n_dim), float(a),
                int(seed), int(iter0), int(n_iter), acc, _stream_ptr(stream, self.device))
        if f_nodes is None:
            self._check(self._lib.ll_pt_run_het(self._h, *tail), "ll_pt_run_het")
        else:
            f_nodes = _host_f64(f_nodes, "f_nodes")
            self._check(self._lib.ll_pt_run_full(self._h, len(f_nodes), f_nodes.ctypes.data_as(C.c_void_p), *tail),
                        "ll_pt_run_full")

    def pt_fused(self, on: bool = True):
        """ll_pt_run_het as one cooperative launch (default) or as 9 launches per iteration"""
        self._check(self._lib.ll_pt_fused(self._h, 1 if on else 0), "ll_pt_fused")

    def pt_swap(self, x, logL, d_h, h_h, betas, u_swap, swapped=None, stream=None):
        n_t, n_w = int(x.shape[0]), int(x.shape[1])
        _shape(x, (n_t, n_w, self.P), "x")
        for v in (logL, d_h, h_h):
            _shape(v, (n_t, n_w), "logL / d_h / h_h")
        _shape(betas, (n_t,), "betas")
        _shape(u_swap, (n_t - 1, n_w), "u_swap")
        _shape(swapped, (n_t - 1, n_w), "swapped")
        self._check(self._lib.ll_pt_swap(self._h, int(x.shape[0]), int(x.shape[1]), _dev_ptr(x, "x"), _dev_ptr(logL, "logL"),
                                         _dev_ptr(d_h, "d_h"), _dev_ptr(h_h, "h_h"), _dev_ptr(betas, "betas"),
                                         _dev_ptr(u_swap, "u_swap"), _dev_ptr_i32(swapped, "swapped"), _stream_ptr(stream, self.device)),
                    "ll_pt_swap")

    def pt_stats(self, logL, d_h, h_h, out3=None, stream=None):
        """-> device tensor [3]: max log L, its index, max extracted SNR"""
        if out3 is None:
            out3 = _torch().empty(3, dtype=_torch().float64, device=logL.device)
        self._check(self._lib.ll_pt_stats(self._h, int(logL.numel()), _dev_ptr(logL, "logL"), _dev_ptr(d_h, "d_h"),
                                          _dev_ptr(h_h, "h_h"), _dev_ptr(out3, "out3"), _stream_ptr(stream, self.device)), "ll_pt_stats")
        return out3

    def het_batch_standin_host(self, params_host, out_host, stream=None):
        n_w = self._check_rows(params_host, out_host)
        ptr = lambda t: None if t is None else C.c_void_p(t.data_ptr() if hasattr(t, "data_ptr") else t.ctypes.data)
        self._check(self._lib.ll_het_batch_standin_host(self._h, n_w, ptr(params_host), ptr(out_host[0]), ptr(out_host[1]),
                                                        ptr(out_host[2]), _stream_ptr(stream, self.device)),
                    "ll_het_batch_standin_host")
        return out_host

    # -- measurement helpers
    def peak_fma(self, which: int, iters: int, stream=None):
        r, ms = C.c_double(), C.c_double()
        self._check(self._lib.ll_peak_fma(self._h, which, iters, C.byref(r), C.byref(ms), _stream_ptr(stream, self.device)), "ll_peak_fma")
        return r.value, ms.value

    def kernel_launches(self) -> int:
        return int(self._lib.ll_kernel_launches(self._h))

    def last_full_stats(self, stream=None):
        a, n = C.c_double(), C.c_int64()
        self._check(self._lib.ll_last_full_stats(self._h, C.byref(a), C.byref(n), _stream_ptr(stream, self.device)), "ll_last_full_stats")
        return a.value, n.value

    def profile_enable(self, on: bool = True):
        self._check(self._lib.ll_profile_enable(self._h, 1 if on else 0), "ll_profile_enable")

    def profile_read(self):
        ms, n = C.c_double(), C.c_int64()
        self._check(self._lib.ll_profile_read(self._h, C.byref(ms), C.byref(n)), "ll_profile_read")
        return ms.value, n.value
