"""CPU oracle — TEST INFRASTRUCTURE ONLY (see the header of ll_oracle.c).

Thin ctypes marshalling over `libll_oracle.so` (built from ll_oracle.c by `oracle.build()` /
`__graft_entry__.build()`).  No arithmetic of the method lives in this file.  Only tests/,
`__graft_entry__.smoke()` and bench.py's cpu_baseline / --impl reference legs may import it; it never
imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libll_oracle.so")
_SRC = os.path.join(_HERE, "ll_oracle.c")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp; plain C, no flags that reorder floating point."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
               "-o", _SO, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
    return _lib


def _p(a: Optional[np.ndarray], dtype=np.float64):
    if a is None:
        return None
    assert a.dtype == dtype and a.flags["C_CONTIGUOUS"], (a.dtype, a.flags)
    return a.ctypes.data_as(C.c_void_p)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with status {rc}")


def n_threads() -> int:
    """Threads the OpenMP loops will use: omp_get_max_threads() (for bench.py's cpu_baseline `cores`)."""
    return int(lib().orc_get_threads())


def set_threads(n: int) -> int:
    """omp_set_num_threads(n) (timing harness: the oracle on one core and on all cores); returns the new count"""
    return int(lib().orc_set_threads(C.c_int(int(n))))


# ------------------------------------------------------------------ spline
def spline_natural(x, y) -> np.ndarray:
    x, y = _f64(x), _f64(y)
    M = np.empty_like(x)
    _check(lib().orc_spline_natural(C.c_int(len(x)), _p(x), _p(y), _p(M)), "spline_natural")
    return M


def set_spline_bc(bc: int) -> None:
    """0 natural (default, reading R1), 1 not-a-knot: process-wide switch of the C oracle (see ll_oracle.c)"""
    _check(lib().orc_set_spline_bc(C.c_int(bc)), "set_spline_bc")


def spline_second_derivatives(x, y) -> np.ndarray:
    """M_j = y''(x_j) under the current boundary condition"""
    x, y = _f64(x), _f64(y)
    M = np.empty_like(x)
    _check(lib().orc_spline_second_derivatives(C.c_int(len(x)), _p(x), _p(y), _p(M)), "spline_second_derivatives")
    return M


def spline_eval(x, y, f_q) -> np.ndarray:
    x, y, f_q = _f64(x), _f64(y), _f64(f_q)
    out = np.empty_like(f_q)
    _check(lib().orc_spline_eval(C.c_int(len(x)), _p(x), _p(y), C.c_int64(f_q.size), _p(f_q), _p(out)), "spline_eval")
    return out


# ------------------------------------------------------------------ stand-in waveform
def standin_fisco(p) -> float:
    p = _f64(p)
    out = C.c_double()
    _check(lib().orc_standin_fisco(_p(p), C.byref(out)), "standin_fisco")
    return out.value


def _n_c_of(P: int, n_m: int) -> int:
    n_c, rem = divmod(P - 5, 2 * n_m)
    assert rem == 0 and n_c in (1, 2, 3), (P, n_m)
    return n_c


def _w_rows(W: np.ndarray, n_c: int) -> int:
    """W [n_f]: one weight row for every channel; W [n_c][n_f]: one row per channel"""
    if W.ndim == 1:
        return 1
    assert W.ndim == 2 and W.shape[0] == n_c, (W.shape, n_c)
    return n_c


def standin_nodes(params, mode_m, c_lm, kappa, f, f_grid_lo, f_grid_hi, n_c=None, split_tc=False):
    """-> amp, phase [n_w][n_m][n_freq], tf [n_w][n_m][n_c][2], band [n_w][2]; n_c from the row length by default.
    split_tc: the phase without its linear term 2 pi f t_c (pass t_shift = params[:, 2] alongside, reading R32)"""
    params, f, c_lm, mode_m = _f64(params), _f64(f), _f64(c_lm), _i32(mode_m)
    n_w, n_m, n = params.shape[0], len(mode_m), len(f)
    n_c = _n_c_of(params.shape[1], n_m) if n_c is None else n_c
    assert params.shape[1] == 5 + 2 * n_c * n_m
    amp = np.empty((n_w, n_m, n))
    phase = np.empty((n_w, n_m, n))
    tf = np.empty((n_w, n_m, n_c, 2))
    band = np.empty((n_w, 2))
    _check(lib().orc_standin_nodes(C.c_int64(n_w), C.c_int(n_m), C.c_int(n_c), _p(mode_m, np.int32), _p(c_lm),
                                   C.c_double(kappa), _p(params), C.c_int(n), _p(f),
                                   C.c_double(f_grid_lo), C.c_double(f_grid_hi), C.c_int(1 if split_tc else 0),
                                   _p(amp), _p(phase), _p(tf), _p(band)), "standin_nodes")
    return amp, phase, tf, band


def standin_direct(p, mode_m, c_lm, kappa, f, f_lo, f_hi, n_c=None) -> np.ndarray:
    """stand-in template of ONE parameter row evaluated directly at f: [n_c][n_freq][2]"""
    p, f, c_lm, mode_m = _f64(p), _f64(f), _f64(c_lm), _i32(mode_m)
    n_m = len(mode_m)
    n_c = _n_c_of(p.shape[0], n_m) if n_c is None else n_c
    assert p.shape == (5 + 2 * n_c * n_m,)
    h = np.empty((n_c, len(f), 2))
    _check(lib().orc_standin_direct(C.c_int(n_m), C.c_int(n_c), _p(mode_m, np.int32), _p(c_lm), C.c_double(kappa),
                                    _p(p), C.c_int64(len(f)), _p(f), C.c_double(f_lo), C.c_double(f_hi), _p(h)),
           "standin_direct")
    return h


# ------------------------------------------------------------------ inner products
def dd(d, W) -> float:
    d, W = _f64(d), _f64(W)
    out = C.c_double()
    _check(lib().orc_dd(C.c_int(d.shape[0]), C.c_int64(d.shape[1]), _p(d), _p(W), C.c_int(_w_rows(W, d.shape[0])),
                        C.byref(out)), "dd")
    return out.value


def inner(a, b, W) -> complex:
    """sum_c sum_k W_k conj(a_k) b_k; the real part is <a|b> (Eq. 3)."""
    a, b, W = _f64(a), _f64(b), _f64(W)
    re, im = C.c_double(), C.c_double()
    _check(lib().orc_inner(C.c_int(a.shape[0]), C.c_int64(a.shape[1]), _p(a), _p(b), _p(W),
                           C.c_int(_w_rows(W, a.shape[0])), C.byref(re), C.byref(im)), "inner")
    return complex(re.value, im.value)


# ------------------------------------------------------------------ full-grid path
def full_batch(f_nodes, amp, phase, tf, band, k_min, df, d, W, want_template=False, t_shift=None):
    """-> dict(logL, d_h, h_h, logL_direct[, h]) for amp/phase [n_w][n_m][n_nodes]; W [n_f] or [n_c][n_f];
    t_shift [n_w] or None: Psi_m(f) = spline_m(f) + 2 pi f t_shift (reading R32)."""
    f_nodes, amp, phase, tf, W = _f64(f_nodes), _f64(amp), _f64(phase), _f64(tf), _f64(W)
    n_w, n_m, n_nodes = amp.shape
    n_c = tf.shape[2]
    n_f = W.shape[-1]
    t_shift = None if t_shift is None else _f64(t_shift)
    assert t_shift is None or t_shift.shape == (n_w,)
    band = None if band is None else _f64(band)
    d = None if d is None else _f64(d)
    out = {k: np.empty(n_w) for k in ("logL", "d_h", "h_h", "logL_direct")}
    h = np.empty((n_c, n_f, 2)) if want_template else None
    _check(lib().orc_full_batch(C.c_int64(n_w), C.c_int(n_m), C.c_int(n_c), C.c_int(n_nodes), _p(f_nodes),
                                _p(amp), _p(phase), _p(tf), _p(band), C.c_int64(n_f), C.c_int64(k_min),
                                C.c_double(df), _p(d), _p(W), C.c_int(_w_rows(W, n_c)), _p(t_shift),
                                _p(out["logL"]), _p(out["d_h"]), _p(out["h_h"]),
                                _p(out["logL_direct"]), _p(h)), "full_batch")
    if want_template:
        out["h"] = h
    return out


def full_batch_tf(f_nodes, amp, phase, tf_nodes, band, k_min, df, d, W, want_template=False, t_shift=None):
    """frequency-dependent transfer function T [n_w][n_m][n_c][n_nodes][2] splined alongside amp/phase (Eq. 8-9)."""
    f_nodes, amp, phase, tf_nodes, W = _f64(f_nodes), _f64(amp), _f64(phase), _f64(tf_nodes), _f64(W)
    n_w, n_m, n_nodes = amp.shape
    n_c = tf_nodes.shape[2]
    assert tf_nodes.shape == (n_w, n_m, n_c, n_nodes, 2)
    n_f = W.shape[-1]
    t_shift = None if t_shift is None else _f64(t_shift)
    assert t_shift is None or t_shift.shape == (n_w,)
    band = None if band is None else _f64(band)
    d = None if d is None else _f64(d)
    out = {k: np.empty(n_w) for k in ("logL", "d_h", "h_h", "logL_direct")}
    h = np.empty((n_c, n_f, 2)) if want_template else None
    _check(lib().orc_full_batch_tf(C.c_int64(n_w), C.c_int(n_m), C.c_int(n_c), C.c_int(n_nodes), _p(f_nodes),
                                   _p(amp), _p(phase), _p(tf_nodes), _p(band), C.c_int64(n_f), C.c_int64(k_min),
                                   C.c_double(df), _p(d), _p(W), C.c_int(_w_rows(W, n_c)), _p(t_shift),
                                   _p(out["logL"]), _p(out["d_h"]), _p(out["h_h"]),
                                   _p(out["logL_direct"]), _p(h)), "full_batch_tf")
    if want_template:
        out["h"] = h
    return out


def tlm_nodes(f_nodes, phase, t_ref) -> np.ndarray:
    """t_lm(f_j) = t_ref - (1/2pi) dphi/df from the natural spline of the node phases (Eq. 8)."""
    f_nodes, phase = _f64(f_nodes), _f64(phase)
    n_w, n_m, n_nodes = phase.shape
    out = np.empty_like(phase)
    _check(lib().orc_tlm_nodes(C.c_int64(n_w), C.c_int(n_m), C.c_int(n_nodes), _p(f_nodes), _p(phase),
                               C.c_double(t_ref), _p(out)), "tlm_nodes")
    return out


def full_batch_standin(wl_modes_m, c_lm, kappa, params, f_nodes, k_min, df, n_f, d, W, want_template=False,
                       split_tc=False):
    """parameters -> node arrays (stand-in, rounded to fp64) -> full_batch.  split_tc: the linear phase term
    2 pi f t_c stays outside the spline (t_shift = t_c, reading R32)."""
    params = _f64(params)
    f_lo, f_hi = float(k_min) * df, float(k_min + n_f - 1) * df
    amp, phase, tf, band = standin_nodes(params, wl_modes_m, c_lm, kappa, f_nodes, f_lo, f_hi, split_tc=split_tc)
    t_shift = np.ascontiguousarray(params[:, 2]) if split_tc else None
    return full_batch(f_nodes, amp, phase, tf, band, k_min, df, d, W, want_template, t_shift=t_shift)


# ------------------------------------------------------------------ heterodyned path
def het_prepare(k_min, df, d, W, h0_dense, f_edges):
    d, W, h0_dense, f_edges = _f64(d), _f64(W), _f64(h0_dense), _f64(f_edges)
    n_c, n_f = d.shape[0], d.shape[1]
    n_b = len(f_edges) - 1
    A0, A1 = np.empty((n_c, n_b, 2)), np.empty((n_c, n_b, 2))
    B0, B1, B2 = np.empty((n_c, n_b)), np.empty((n_c, n_b)), np.empty((n_c, n_b))
    ddb = C.c_double()
    _check(lib().orc_het_prepare(C.c_int(n_c), C.c_int64(n_f), C.c_int64(k_min), C.c_double(df), _p(d), _p(W),
                                 C.c_int(_w_rows(W, n_c)), _p(h0_dense), C.c_int(len(f_edges)), _p(f_edges),
                                 _p(A0), _p(A1), _p(B0), _p(B1), _p(B2), C.byref(ddb)), "het_prepare")
    return dict(A0=A0, A1=A1, B0=B0, B1=B1, B2=B2, dd_band=ddb.value)


def het_batch(f_edges, amp_e, phase_e, tf, h0_edges, summ, t_shift=None):
    """t_shift [n_w] or None: Psi_m(f_e) = phase_e + 2 pi f_e t_shift (reading R32)"""
    f_edges, amp_e, phase_e, tf, h0_edges = _f64(f_edges), _f64(amp_e), _f64(phase_e), _f64(tf), _f64(h0_edges)
    n_w, n_m, n_e = amp_e.shape
    n_c = tf.shape[2]
    t_shift = None if t_shift is None else _f64(t_shift)
    assert t_shift is None or t_shift.shape == (n_w,)
    out = {k: np.empty(n_w) for k in ("logL", "d_h", "h_h")}
    _check(lib().orc_het_batch(C.c_int64(n_w), C.c_int(n_m), C.c_int(n_c), C.c_int(n_e), _p(f_edges),
                               _p(amp_e), _p(phase_e), _p(tf), _p(t_shift), _p(h0_edges),
                               _p(_f64(summ["A0"])), _p(_f64(summ["A1"])), _p(_f64(summ["B0"])), _p(_f64(summ["B1"])),
                               C.c_double(summ["dd_band"]), _p(out["logL"]), _p(out["d_h"]), _p(out["h_h"])),
           "het_batch")
    return out


def het_batch_standin(mode_m, c_lm, kappa, params, f_edges, h0_edges, summ, chunk=8192):
    """parameters -> amp/phase at the edges (stand-in evaluated directly, no spline) -> het_batch."""
    params = _f64(params)
    outs = []
    for lo in range(0, params.shape[0], chunk):
        amp, phase, tf, _ = standin_nodes(params[lo:lo + chunk], mode_m, c_lm, kappa, f_edges,
                                          float(f_edges[0]), float(f_edges[-1]))
        outs.append(het_batch(f_edges, amp, phase, tf, h0_edges, summ))
    if not outs:
        return {k: np.empty(0) for k in ("logL", "d_h", "h_h")}
    return {k: np.concatenate([o[k] for o in outs]) for k in outs[0]}
