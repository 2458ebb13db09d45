"""CPU oracle, part 4 — TEST INFRASTRUCTURE ONLY (never imported by the product path; imports nothing of it).

Full-grid likelihood with PER-WALKER node grids: each walker's sparse nodes span its own
band instead of one shared grid.  Nothing new is computed: it is the full-grid oracle (oracle.full_batch: natural
cubic spline of amplitude and phase in f, Eq. 7, 9, 3, 2; readings R1, R2, R6-R8) applied to one walker at a time
with that walker's own nodes.

Reading R30: a spline is not extrapolated beyond its own nodes — the template of walker w is zero
outside [x_{w,0}, x_{w,n-1}] (intersected with the caller's band, if one is given; bounds inclusive), which is what
"each walker's nodes spanning its own [f_min, f_max]" means for the band mask of reading R10.

Pins (tests/test_oracle_pins.py): identical to the shared-node oracle when every walker has the same nodes and the
band is the node span; SciPy natural spline + numpy complex sums per walker on a tiny grid with different nodes
per walker; a template that is a single global cubic in amplitude and linear in phase does not depend on where the
interior nodes are.
"""
from __future__ import annotations

import numpy as np

import oracle as orc


def full_batch_pw(f_nodes_w, amp, phase, tf, band, k_min, df, d, W, t_shift=None):
    """f_nodes_w [n_w][n_nodes]; amp, phase [n_w][n_m][n_nodes]; tf [n_w][n_m][n_c][2]; band [n_w][2] or None;
    W [n_f] or [n_c][n_f]; t_shift [n_w] or None (linear phase term outside the spline, reading R32)."""
    f_nodes_w = np.asarray(f_nodes_w, dtype=np.float64)
    n_w = f_nodes_w.shape[0]
    out = {k: np.empty(n_w) for k in ("logL", "d_h", "h_h", "logL_direct")}
    for w in range(n_w):
        x = np.ascontiguousarray(f_nodes_w[w])
        lo, hi = x[0], x[-1]
        if band is not None:
            lo, hi = max(lo, band[w][0]), min(hi, band[w][1])
        r = orc.full_batch(x, amp[w:w + 1], phase[w:w + 1], tf[w:w + 1], np.array([[lo, hi]]), k_min, df, d, W,
                           t_shift=None if t_shift is None else np.asarray(t_shift, dtype=np.float64)[w:w + 1])
        for k in out:
            out[k][w] = r[k][0]
    return out
