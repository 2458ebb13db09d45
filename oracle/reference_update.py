"""CPU oracle, part 2 — TEST INFRASTRUCTURE ONLY (never imported by the product path; imports nothing of it).

The two steps the paper wraps around the heterodyned likelihood inside the sampling loop, written out with numpy
on top of the C oracle's primitives (oracle.standin_direct / inner / dd / het_prepare / standin_fisco):

  reference update   "The reference template is updated every 5000 iterations of the sampler by replacing it with
                     the highest Likelihood point in the population."
                     "The frequency content contained in the reference template ... is set as the frequency band
                     over which the Heterodyning method is applied (h0(f) != 0)."
  audit              "the brute-force Likelihood can ... verify the Heterodyning results"

Readings: R12 edge placement geomspace(f_0, min(f_last, f_ISCO(best)), n_e) with exact end points;
R13 bin membership [e_b, e_{b+1}), last closed, so the heterodyne bins cover the dense bins with
e_0 <= f_i <= e_last; ties of the maximum go to the lowest index; non-finite log L never wins.

Pins (tests/test_oracle_pins.py): the audit at h = d is -1/2 <d-h|d-h> = 0 bit for bit in the direct residual
form and |.| <= 1e-6 in the three-term form; audit == heterodyne at h = h0 after an update; the edges equal
numpy.geomspace; the best index equals a pure-Python scan.
"""
from __future__ import annotations

import numpy as np

import oracle as orc


def best_walker(logL) -> int:
    """index of the largest finite log L, lowest index on ties; -1 if none is finite"""
    best, bi = -np.inf, -1
    for i, x in enumerate(np.asarray(logL, dtype=np.float64)):
        if np.isfinite(x) and (bi < 0 or x > best):
            best, bi = float(x), i
    return bi


def reference_edges(p_best, f_first: float, f_last: float, n_edges: int) -> np.ndarray:
    """reading R12: log-spaced edges over the band where the reference has its untapered support"""
    f_top = min(f_last, orc.standin_fisco(p_best))
    if not f_top > f_first:
        raise ValueError("the best walker's f_ISCO lies below the grid: no heterodyne band")
    e = np.geomspace(f_first, f_top, n_edges)
    e[0], e[-1] = f_first, f_top
    return e


def reference_update(params, logL, mode_m, c_lm, kappa, k_min, df, n_f, d, W, n_edges):
    """-> dict(best, f_edges, h0, h0_edges, summ): the new reference and its summary data (Eq. 15-19)"""
    f = (k_min + np.arange(n_f, dtype=np.int64)).astype(np.float64) * df
    bi = best_walker(logL)
    if bi < 0:
        raise ValueError("no finite log L in the population")
    p = np.asarray(params, dtype=np.float64)[bi]
    e = reference_edges(p, float(f[0]), float(f[-1]), n_edges)
    h0 = orc.standin_direct(p, mode_m, c_lm, kappa, f, float(f[0]), float(f[-1]))
    h0e = orc.standin_direct(p, mode_m, c_lm, kappa, e, float(f[0]), float(f[-1]))
    summ = orc.het_prepare(k_min, df, d, W, h0, e)
    return {"best": bi, "f_edges": e, "h0": h0, "h0_edges": h0e, "summ": summ}


def audit(params, mode_m, c_lm, kappa, k_min, df, n_f, d, W, f_edges):
    """dense log L of every row over the dense bins the heterodyne bins cover, template evaluated directly at each
    bin; three-term form log L = <d|h> - 1/2 <h|h> - 1/2 <d|d>_band (Eq. 2-3).  Also returns the direct residual
    form -1/2 sum W |d-h|^2 (reading R8)."""
    f = (k_min + np.arange(n_f, dtype=np.int64)).astype(np.float64) * df
    m = (f >= f_edges[0]) & (f <= f_edges[-1])
    fm, Wm = np.ascontiguousarray(f[m]), np.ascontiguousarray(np.asarray(W)[..., m])   # W [n_f] or [n_c][n_f]
    dm = np.ascontiguousarray(np.asarray(d)[:, m, :])
    ddb = orc.dd(dm, Wm)
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    out = {k: np.empty(params.shape[0]) for k in ("logL", "d_h", "h_h", "logL_direct")}
    for w, p in enumerate(params):
        h = orc.standin_direct(p, mode_m, c_lm, kappa, fm, float(f[0]), float(f[-1]))
        out["d_h"][w] = orc.inner(dm, h, Wm).real
        out["h_h"][w] = orc.inner(h, h, Wm).real
        out["logL"][w] = out["d_h"][w] - 0.5 * out["h_h"][w] - 0.5 * ddb
        r = dm - h
        out["logL_direct"][w] = -0.5 * float(np.sum((Wm if Wm.ndim == 2 else Wm[None, :]) * (r[..., 0] ** 2 + r[..., 1] ** 2)))
    return out
