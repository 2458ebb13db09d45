"""Finish a seeded workload (workloads.py) with the CUDA library itself and load it into a Context.

The recipe has two stages that need a template: the luminosity scale that puts the injection at
SNR 500 (reading R18) and the data stream d = h_inj + n (R19).  Here both come from the library's own kernels
(`ll_full_batch_standin` with d = 0 for <h|h>, `ll_full_template_standin` / `ll_template_standin` for h_inj), so
bench.py never touches oracle/ for its inputs.  The tests do the same two stages with the oracle instead and
hand the same arrays to both sides.
"""
from __future__ import annotations

import math

import numpy as np
import torch

from . import workloads as wlm
from .binding import Context, LL_PREC_FP64


def _dev(a, device):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device=device)


def make_context(wl: wlm.Workload, precision: int = LL_PREC_FP64, device=None) -> Context:
    ctx = Context(n_modes=wl.n_m, precision=precision, device=device, n_channels=wl.n_c)
    ctx.standin_config(wl.modes_l, wl.modes_m, wl.c_lm, wl.kappa)
    return ctx


def setup_full(ctx: Context, wl: wlm.Workload):
    """config 0 / 2 recipe: data = spline-path template of the injection (+ noise).  Returns device tensors."""
    dev = f"cuda:{ctx.device}"
    g = wl.grid
    W = _dev(wl.W, dev)
    zero = torch.zeros((wl.n_c, g.n_f, 2), dtype=torch.float64, device=dev)
    ctx.set_data(g.n_f, g.k_min, g.df, zero, W)
    if not wl.finished:
        inj = _dev(wl.inj[None, :], dev)
        _, _, hh = ctx.full_batch_standin(wl.f_nodes, inj)
        wl.finish_distance(float(hh.cpu()[0]))
    h = ctx.full_template_standin(wl.f_nodes, wl.inj)
    d = h if wl.noise is None else h + _dev(wl.noise, dev)
    d = d.contiguous()
    ctx.set_data(g.n_f, g.k_min, g.df, d, W)
    return dict(d=d, W=W, params=_dev(wl.params, dev))


def setup_het(ctx: Context, wl: wlm.Workload):
    """config 1 / 3 / 4 recipe: h0 = directly evaluated template of the injection on the dense grid and at the
    edges; data = h0 + noise; summary data from ll_het_prepare."""
    dev = f"cuda:{ctx.device}"
    g = wl.grid
    f = _dev(g.freqs(), dev)
    W = _dev(wl.W, dev)
    f_lo, f_hi = float(g.k_min * g.df), float(g.k_max * g.df)
    if not wl.finished:
        h1 = ctx.template_standin(wl.inj, f, f_lo, f_hi)
        ctx.set_data(g.n_f, g.k_min, g.df, h1, W)                       # <h|h> = <d|d> of d := h (F0 kernel)
        wl.finish_distance(ctx.get_dd()[0])
    h0 = ctx.template_standin(wl.inj, f, f_lo, f_hi)
    d = h0 if wl.noise is None else h0 + _dev(wl.noise, dev)
    d = d.contiguous()
    ctx.set_data(g.n_f, g.k_min, g.df, d, W)
    h0e = ctx.template_standin(wl.inj, _dev(wl.f_edges, dev), f_lo, f_hi)
    ctx.het_prepare(wl.f_edges, h0, h0e)
    return dict(d=d, W=W, h0=h0, h0_edges=h0e, params=_dev(wl.params, dev))


def setup(ctx: Context, wl: wlm.Workload):
    return setup_full(ctx, wl) if wl.path == "full" else setup_het(ctx, wl)


def smooth_tf_nodes(params, f_nodes, n_m: int = 1, n_c: int = 2):
    """A smooth frequency-dependent transfer function at the nodes for timing / demonstration runs of
    ll_full_batch_tf: T^c_m(f_j) = T^c_m(params) * (1 + 0.2 x_j) e^{2 i x_j}, x = log(f/f_0)/log(f_last/f_0).
    (The physical response's formula is in the paper's ref. [44], not in PAPER.md; any smooth T exercises the
    same six-spline path.)  Returns a device tensor [n_w][n_m][n_c][n_nodes][2]."""
    dev = params.device
    f = torch.as_tensor(np.asarray(f_nodes, dtype=np.float64), device=dev)
    x = torch.log(f / f[0]) / math.log(float(f_nodes[-1]) / float(f_nodes[0]))
    mod = (1.0 + 0.2 * x)
    cr, ci = mod * torch.cos(2.0 * x), mod * torch.sin(2.0 * x)
    t = params[:, 5:5 + 2 * n_c * n_m].reshape(-1, n_m, n_c, 1, 2)
    tr, ti = t[..., 0], t[..., 1]
    out = torch.stack([tr * cr - ti * ci, tr * ci + ti * cr], dim=-1)
    return out.contiguous()
