"""Pins for the CPU oracle (oracle/ll_oracle.c) against things OTHER than itself:
library routines (SciPy CubicSpline, numpy.linalg), closed forms, textbook numbers, invariants the
paper states, and brute force written a different way (numpy complex arithmetic, math.fsum, mpmath).
All CPU-only (-m "not gpu").  Citations: PAPER.md line numbers; R<n> = DESIGN.md §3 readings.
"""
import math

import mpmath
import numpy as np
import pytest
from scipy.interpolate import CubicSpline

from paper_2111_01064_b200 import workloads as wlm

TWO_PI = 2.0 * math.pi


# --------------------------------------------------------------------------- helpers (independent formulation)
def _brute_full(f_nodes, amp, phase, tf, band, k_min, df, d, W):
    """SciPy natural spline + numpy complex arithmetic + math.fsum.  One walker at a time."""
    n_w, n_m, _ = amp.shape
    n_c = tf.shape[2]
    n_f = W.shape[0]
    f = np.arange(k_min, k_min + n_f, dtype=np.float64) * df
    dc = d[..., 0] + 1j * d[..., 1]
    out = {k: np.zeros(n_w) for k in ("logL", "d_h", "h_h")}
    dd = math.fsum((W[None, :] * np.abs(dc) ** 2).ravel())
    for w in range(n_w):
        mask = np.ones(n_f, bool) if band is None else (f >= band[w, 0]) & (f <= band[w, 1])
        h = np.zeros((n_c, n_f), complex)
        for m in range(n_m):
            A = CubicSpline(f_nodes, amp[w, m], bc_type="natural")(f)
            P = CubicSpline(f_nodes, phase[w, m], bc_type="natural")(f)
            hm = A * np.exp(-1j * P)
            for c in range(n_c):
                h[c] += (tf[w, m, c, 0] + 1j * tf[w, m, c, 1]) * hm
        h[:, ~mask] = 0.0
        out["d_h"][w] = math.fsum((W[None, :] * (np.conj(dc) * h).real).ravel())
        out["h_h"][w] = math.fsum((W[None, :] * np.abs(h) ** 2).ravel())
        out["logL"][w] = out["d_h"][w] - 0.5 * out["h_h"][w] - 0.5 * dd
    return out


def _rand_smooth_nodes(rng, n_w, n_m, f_nodes):
    """Smooth random amp/phase node arrays with a LISA-like dynamic range (phase ~1e3 rad)."""
    x = np.log(f_nodes / f_nodes[0])
    amp = np.empty((n_w, n_m, len(f_nodes)))
    ph = np.empty_like(amp)
    for w in range(n_w):
        for m in range(n_m):
            a, b, c = rng.uniform(0.5, 2.0), rng.uniform(-1, 1), rng.uniform(-300, 300)
            amp[w, m] = a * np.exp(-0.7 * x) * (1.0 + 0.1 * np.sin(b + x))
            ph[w, m] = c * x + 40.0 * np.cos(0.3 * x + b) + 900.0 * f_nodes / f_nodes[-1]
    return amp, ph


def _unit_tf(rng, n_w, n_m, n_c=2):
    ang = rng.uniform(0, TWO_PI, (n_w, n_m, n_c))
    return np.stack([np.cos(ang), np.sin(ang)], axis=-1)


def _c(a):
    return a[..., 0] + 1j * a[..., 1]


# --------------------------------------------------------------------------- spline (R1, R21)
@pytest.mark.parametrize("n", [3, 4, 7, 16, 257])
def test_spline_matches_scipy_natural(orc, n):
    rng = np.random.default_rng(n)
    x = np.sort(rng.uniform(1e-4, 5e-2, n))
    x[0], x[-1] = 1e-4, 5e-2
    y = rng.standard_normal(n).cumsum()
    cs = CubicSpline(x, y, bc_type="natural")
    M = orc.spline_natural(x, y)
    np.testing.assert_allclose(M, cs(x, 2), rtol=1e-10, atol=1e-10 * np.abs(cs(x, 2)).max())
    assert M[0] == 0.0 and M[-1] == 0.0
    q = rng.uniform(x[0], x[-1], 500)
    np.testing.assert_allclose(orc.spline_eval(x, y, q), cs(q), rtol=0, atol=1e-12 * np.abs(y).max())


def test_spline_dense_gaussian_elimination(orc):
    """The tridiagonal system of R1 solved as a dense matrix (numpy.linalg.solve)."""
    rng = np.random.default_rng(1)
    for n in (3, 5, 12, 16):
        x = np.cumsum(rng.uniform(0.1, 1.0, n))
        y = rng.standard_normal(n)
        h = np.diff(x)
        A = np.zeros((n, n))
        r = np.zeros(n)
        A[0, 0] = A[-1, -1] = 1.0
        for j in range(1, n - 1):
            A[j, j - 1], A[j, j], A[j, j + 1] = h[j - 1] / 6, (h[j - 1] + h[j]) / 3, h[j] / 6
            r[j] = (y[j + 1] - y[j]) / h[j] - (y[j] - y[j - 1]) / h[j - 1]
        np.testing.assert_allclose(orc.spline_natural(x, y), np.linalg.solve(A, r), rtol=1e-11, atol=1e-12)


def test_spline_reproduces_linear_and_interpolates_nodes(orc):
    x = wlm.geomspace_exact(1e-4, 5e-2, 64)
    y = 3.0e6 * x - 17.0                      # 2 pi f t_c like term: any cubic spline is exact (R2)
    q = np.linspace(x[0], x[-1], 1001)
    np.testing.assert_allclose(orc.spline_eval(x, y, q), 3.0e6 * q - 17.0, rtol=0, atol=1e-10)
    np.testing.assert_allclose(orc.spline_natural(x, y), 0.0, atol=1e-3)  # |M| ~ rounding of y / h^2
    y2 = np.sin(200 * x) + x ** -0.5
    np.testing.assert_allclose(orc.spline_eval(x, y2, x), y2, rtol=1e-15, atol=0)


def test_spline_c2_continuity_and_clamped_lookup(orc):
    rng = np.random.default_rng(5)
    x = np.cumsum(rng.uniform(0.5, 1.5, 9))
    y = rng.standard_normal(9)
    eps = 1e-6
    for xi in x[1:-1]:
        lo, mid, hi = orc.spline_eval(x, y, [xi - eps, xi, xi + eps])
        # value and first derivative continuous: symmetric difference is O(eps^2)
        assert abs(hi - 2 * mid + lo) < 1e-9
    M = orc.spline_natural(x, y)
    # second derivative is piecewise linear between the M_j: midpoint value equals the mean
    xm = 0.5 * (x[:-1] + x[1:])
    e2 = 1e-4
    num2 = (orc.spline_eval(x, y, xm + e2) - 2 * orc.spline_eval(x, y, xm) + orc.spline_eval(x, y, xm - e2)) / e2 ** 2
    np.testing.assert_allclose(num2, 0.5 * (M[:-1] + M[1:]), atol=1e-6)
    # a query exactly on the last node uses the last interval (clamp, R21)
    assert orc.spline_eval(x, y, [x[-1]])[0] == pytest.approx(y[-1], abs=1e-14)


# --------------------------------------------------------------------------- stand-in waveform (R9)
def _row(mc_msun=3e5, q=0.5, t_c=7.0e4, phi_c=1.2, inv_d=1.0, n_m=1, ang=None):
    p = np.zeros(5 + 4 * n_m)
    p[:5] = [mc_msun * wlm.GMSUN_S, q, t_c, phi_c, inv_d]
    ang = np.linspace(0.3, 2.9, 2 * n_m) if ang is None else ang
    p[5::2], p[6::2] = np.cos(ang), np.sin(ang)
    return p


def test_fisco_textbook_number(orc):
    """f_ISCO = c^3/(6^{3/2} pi G M) = 4397 Hz for M = 1 Msun (textbook, ~4.4 kHz Msun/M)."""
    p = _row(mc_msun=0.25 ** 0.6, q=1.0)      # eta = 1/4 -> M = Mc eta^{-3/5} = 1 Msun
    assert orc.standin_fisco(p) == pytest.approx(4397.0, rel=2e-4)
    # scales as 1/M
    p2 = _row(mc_msun=1e6 * 0.25 ** 0.6, q=1.0)
    assert orc.standin_fisco(p2) == pytest.approx(orc.standin_fisco(p) / 1e6, rel=1e-14)


def test_standin_phase_derivative_is_newtonian_chirp_time(orc):
    """(1/2pi) dPsi/df = t_c - tau(f),  tau = (5/256) Mc^{-5/3} (pi f)^{-8/3}  (Peters' time to coalescence).
    Fails on a wrong sign or power in the PN term, a wrong eta/M relation, or a missing 2 pi f t_c."""
    p = _row(mc_msun=4e5, q=0.3, t_c=9.0e4)
    mc = p[0]
    f = np.array([2e-4, 5e-4, 1e-3, 3e-3])
    hstep = f * 1e-5
    kw = dict(mode_m=[2], c_lm=[1.0], kappa=0.5, f_grid_lo=0.0, f_grid_hi=1.0)
    _, php, _, _ = orc.standin_nodes(p[None], f=f + hstep, **kw)
    _, phm, _, _ = orc.standin_nodes(p[None], f=f - hstep, **kw)
    t_of_f = (php[0, 0] - phm[0, 0]) / (2 * hstep) / TWO_PI
    tau = 5.0 / 256.0 * mc ** (-5.0 / 3.0) * (math.pi * f) ** (-8.0 / 3.0)
    np.testing.assert_allclose(p[2] - t_of_f, tau, rtol=1e-6)


def test_standin_q_enters_phase_only_through_fisco(orc):
    """eta v^5 = (pi Mc f)^{5/3}: at fixed chirp mass the phase is independent of q."""
    f = wlm.geomspace_exact(1e-4, 2e-3, 40)
    kw = dict(mode_m=[2], c_lm=[1.0], kappa=0.5, f=f, f_grid_lo=0.0, f_grid_hi=1.0)
    _, ph1, _, b1 = orc.standin_nodes(_row(q=0.2)[None], **kw)
    _, ph2, _, b2 = orc.standin_nodes(_row(q=0.9)[None], **kw)
    np.testing.assert_allclose(ph1, ph2, rtol=0, atol=1e-9 * np.abs(ph1).max())
    assert b1[0, 1] != b2[0, 1]


def test_standin_amplitude_powerlaw_and_taper(orc):
    p = _row(mc_msun=5e5, q=1.0, inv_d=2.0)
    fi = orc.standin_fisco(p)
    kw = dict(mode_m=[2], c_lm=[1.0], kappa=0.5, f_grid_lo=0.0, f_grid_hi=1.0)
    f = np.array([0.1, 0.5, 1.0]) * fi
    a, _, _, band = orc.standin_nodes(p[None], f=f, **kw)
    np.testing.assert_allclose(a[0, 0], 2.0 * f ** (-7.0 / 6.0), rtol=1e-14)          # untapered below f_ISCO
    assert band[0, 1] == pytest.approx(1.5 * fi, rel=1e-15)
    # taper: 1/2 at the midpoint, 0 at and beyond (1+kappa) f_ISCO, smooth (C^2) at both ends
    f2 = np.array([1.25, 1.5, 1.7]) * fi
    a2, _, _, _ = orc.standin_nodes(p[None], f=f2, **kw)
    np.testing.assert_allclose(a2[0, 0] / (2.0 * f2 ** (-7.0 / 6.0)), [0.5, 0.0, 0.0], atol=1e-15)
    for x0 in (1.0, 1.5):
        e = 1e-4
        fx = np.array([x0 - 2 * e, x0 - e, x0, x0 + e, x0 + 2 * e]) * fi
        t = orc.standin_nodes(p[None], f=fx, **kw)[0][0, 0] / (2.0 * fx ** (-7.0 / 6.0))
        assert abs(t[1] - 2 * t[2] + t[3]) / e ** 2 < 1e-2 * 60   # second derivative -> 0 (s^3 factor), not O(1)/kappa^2
        assert abs((t[3] - t[1]) / (2 * e)) < 1e-3
    # monotone on the taper
    fx = np.linspace(1.0, 1.5, 50) * fi
    t = orc.standin_nodes(p[None], f=fx, **kw)[0][0, 0] / (2.0 * fx ** (-7.0 / 6.0))
    assert np.all(np.diff(t) <= 1e-15)


def test_standin_mode_relation(orc):
    """Psi_lm(f) = (m/2) Psi_22(2f/m);  A_lm(f) = c_lm f^{-7/6}/D taper(2f/(m f_ISCO))  (BASELINE config 3)."""
    p6 = _row(n_m=3)
    p1 = np.concatenate([p6[:5], p6[5:9]])
    f = wlm.geomspace_exact(2e-4, 3e-3, 17)
    kw = dict(kappa=0.5, f_grid_lo=0.0, f_grid_hi=1.0)
    a, ph, tf, band = orc.standin_nodes(p6[None], mode_m=[2, 1, 3], c_lm=[1.0, 0.3, 0.2], f=f, **kw)
    for i, (m, c) in enumerate([(2, 1.0), (1, 0.3), (3, 0.2)]):
        a22, ph22, _, _ = orc.standin_nodes(p1[None], mode_m=[2], c_lm=[1.0], f=2 * f / m, **kw)
        np.testing.assert_allclose(ph[0, i], (m / 2) * ph22[0, 0], rtol=1e-15)
        # amplitude: same taper argument as the (2,2) mode at 2f/m, power law taken at f
        np.testing.assert_allclose(a[0, i], c * a22[0, 0] * (f / (2 * f / m)) ** (-7.0 / 6.0), rtol=1e-14)
    assert tf.shape == (1, 3, 2, 2) and np.all(tf.ravel() == p6[5:])
    assert band[0, 1] == pytest.approx(1.5 * orc.standin_fisco(p6) * 1.5, rel=1e-15)  # max m/2 = 3/2


# --------------------------------------------------------------------------- <h|h> closed form (Eq. 3)
def _flat_setup(orc, t_obs, n_nodes, S0=3.0e-40):
    grid = wlm.make_grid(t_obs)
    f = grid.freqs()
    w = np.ones(grid.n_f)
    w[0] = w[-1] = 0.5
    W = 4.0 * grid.df * w / S0
    p = _row(mc_msun=50.0, q=1.0, t_c=0.6 * t_obs, inv_d=1.0)   # f_ISCO ~ 50 Hz >> band: no taper
    assert orc.standin_fisco(p) > 1.0
    return grid, f, W, p, S0


def test_hh_closed_form_flat_psd_direct(orc):
    """<h|h> = (6/(D^2 S0)) (f_lo^{-4/3} - f_hi^{-4/3}) for |T^A| = |T^E| = 1, no taper, flat PSD.
    The discrete trapezoid sum differs from the integral by the Euler-Maclaurin term
    (df^2/12)[g'(f_hi) - g'(f_lo)], g = f^{-7/3}; after adding it the residual is ~1e-6 (cfg-0 grid)."""
    grid, f, W, p, S0 = _flat_setup(orc, 2.0 ** 17, 0)
    h = orc.standin_direct(p, [2], [1.0], 0.5, f, f[0], f[-1])
    hh = orc.inner(h, h, W).real
    flo, fhi = f[0], f[-1]
    integral = 6.0 / S0 * (flo ** (-4.0 / 3.0) - fhi ** (-4.0 / 3.0))
    gp = lambda x: -7.0 / 3.0 * x ** (-10.0 / 3.0)
    em = 8.0 / S0 * grid.df ** 2 / 12.0 * (gp(fhi) - gp(flo))
    assert hh == pytest.approx(integral, rel=2e-3)
    assert abs(hh - integral) / integral > 5e-4            # the trapezoid bias is really there (+1.3e-3)
    assert hh == pytest.approx(integral + em, rel=5e-6)
    # exact discrete sum with mpmath (50 digits)
    mpmath.mp.dps = 50
    s = mpmath.fsum(mpmath.mpf(float(Wk)) * mpmath.mpf(float(fk)) ** (mpmath.mpf(-7) / 3) for Wk, fk in zip(W, f))
    assert hh == pytest.approx(float(2 * s), rel=1e-14)


def test_hh_closed_form_through_spline_path(orc):
    grid, f, W, p, S0 = _flat_setup(orc, 2.0 ** 17, 256)
    f_nodes = wlm.geomspace_exact(1e-4, 0.05, 256)
    r = orc.full_batch_standin([2], [1.0], 0.5, p[None], f_nodes, grid.k_min, grid.df, grid.n_f, None, W)
    flo, fhi = f[0], f[-1]
    integral = 6.0 / S0 * (flo ** (-4.0 / 3.0) - fhi ** (-4.0 / 3.0))
    gp = lambda x: -7.0 / 3.0 * x ** (-10.0 / 3.0)
    em = 8.0 / S0 * grid.df ** 2 / 12.0 * (gp(fhi) - gp(flo))
    assert r["h_h"][0] == pytest.approx(integral + em, rel=2e-4)     # spline amplitude error <= 7e-5 (natural BC)
    # 1024 nodes on the cfg-1 grid: 1e-5
    grid2, f2, W2, p2, _ = _flat_setup(orc, 2.0 ** 22, 1024)
    f_nodes2 = wlm.geomspace_exact(1e-4, 0.05, 1024)
    r2 = orc.full_batch_standin([2], [1.0], 0.5, p2[None], f_nodes2, grid2.k_min, grid2.df, grid2.n_f, None, W2)
    integral2 = 6.0 / S0 * (f2[0] ** (-4.0 / 3.0) - f2[-1] ** (-4.0 / 3.0))
    assert r2["h_h"][0] == pytest.approx(integral2, rel=1e-5)


# --------------------------------------------------------------------------- log L invariants (Eq. 2)
@pytest.fixture(scope="module")
def cfg0(orc):
    wl = wlm.make_workload(0)
    g = wl.grid
    run = lambda params, d, tmpl=False: orc.full_batch_standin(
        wl.modes_m, wl.c_lm, wl.kappa, params, wl.f_nodes, g.k_min, g.df, g.n_f, d, wl.W, want_template=tmpl)
    wl.finish_distance(run(wl.inj[None], None)["h_h"][0])
    h = run(wl.inj[None], None, True)["h"]
    d = wl.make_data(h)
    return wl, d, run


def test_logL_zero_at_truth_noiseless(cfg0):
    """noiseless data, correct model => the maximum log L = 0 at Theta_true."""
    wl, d, run = cfg0
    r = run(wl.params, d)
    assert abs(r["logL"][0]) <= 1e-6
    assert abs(r["logL_direct"][0]) <= 1e-20
    assert math.sqrt(r["h_h"][0]) == pytest.approx(500.0, rel=1e-12)        # R18
    assert np.all(r["logL"][1:] < -1.0)
    np.testing.assert_allclose(r["logL"], r["logL_direct"], rtol=1e-9, atol=1e-6)   # R8: both forms of Eq. 2
    # Cauchy-Schwarz: <d|h>^2 <= <d|d><h|h>
    dd = -2.0 * r["logL"] + 2.0 * r["d_h"] - r["h_h"]
    assert np.all(r["d_h"] ** 2 <= dd * r["h_h"] * (1 + 1e-12))


def test_scaling_laws(cfg0):
    """d_h ∝ 1/D, h_h ∝ 1/D^2; phi_c -> phi_c + delta rotates the complex overlap, h_h unchanged."""
    wl, d, run = cfg0
    p = wl.params[:8].copy()
    r0 = run(p, d)
    p2 = p.copy(); p2[:, 4] *= 3.0
    r2 = run(p2, d)
    np.testing.assert_allclose(r2["d_h"], 3.0 * r0["d_h"], rtol=1e-13)
    np.testing.assert_allclose(r2["h_h"], 9.0 * r0["h_h"], rtol=1e-13)
    # overlap O = sum W conj(d) h ; h(phi_c + delta) = e^{+i delta} h  => Re part rotates
    delta = 0.7
    p3 = p.copy(); p3[:, 3] += delta
    p4 = p.copy(); p4[:, 3] += math.pi / 2
    r3, r4 = run(p3, d), run(p4, d)
    re, im = r0["d_h"], r4["d_h"]               # Re O and Re(i O) = -Im O
    np.testing.assert_allclose(r3["d_h"], re * math.cos(delta) + im * math.sin(delta), rtol=1e-9, atol=1e-7)
    np.testing.assert_allclose(r3["h_h"], r0["h_h"], rtol=1e-13)
    # maximising over 1/D analytically: max_D log L = d_h^2/(2 h_h) - dd/2 >= log L
    dd = -2.0 * r0["logL"] + 2.0 * r0["d_h"] - r0["h_h"]
    assert np.all(0.5 * r0["d_h"] ** 2 / r0["h_h"] - 0.5 * dd >= r0["logL"] - 1e-9)


# --------------------------------------------------------------------------- brute force, tiny inputs
@pytest.mark.parametrize("n_m,n_nodes,n_f,banded", [(1, 4, 16, False), (1, 8, 64, True), (3, 6, 33, True)])
def test_full_path_brute_force_tiny(orc, n_m, n_nodes, n_f, banded):
    rng = np.random.default_rng(100 + n_nodes)
    k_min, df = 5, 1.0 / 4096.0
    f_lo, f_hi = k_min * df, (k_min + n_f - 1) * df
    f_nodes = wlm.geomspace_exact(f_lo * 0.9, f_hi * 1.05, n_nodes)
    amp, ph = _rand_smooth_nodes(rng, 3, n_m, f_nodes)
    tf = _unit_tf(rng, 3, n_m) * rng.uniform(0.5, 1.5, (3, n_m, 2, 1))
    W = rng.uniform(0.5, 2.0, n_f)
    d = rng.standard_normal((2, n_f, 2))
    band = None
    if banded:
        band = np.array([[f_lo, f_hi], [f_lo + 3.2 * df, f_hi - 5.5 * df], [f_hi * 2, f_hi * 3]])
    o = orc.full_batch(f_nodes, amp, ph, tf, band, k_min, df, d, W)
    b = _brute_full(f_nodes, amp, ph, tf, band, k_min, df, d, W)
    for k in ("logL", "d_h", "h_h"):
        np.testing.assert_allclose(o[k], b[k], rtol=1e-11, atol=1e-11)
    if banded:      # a band that misses the grid gives log L = -<d|d>/2 (include/ll.h)
        assert o["h_h"][2] == 0.0 and o["d_h"][2] == 0.0
        assert o["logL"][2] == pytest.approx(-0.5 * orc.dd(d, W), rel=1e-15)


def test_full_path_mpmath_one_walker(orc):
    """One (walker, 2 modes) case summed with 40-digit arithmetic on top of SciPy spline values."""
    rng = np.random.default_rng(7)
    k_min, df, n_f = 3, 1.0 / 512.0, 12
    f = np.arange(k_min, k_min + n_f) * df
    f_nodes = wlm.geomspace_exact(f[0], f[-1], 5)
    amp, ph = _rand_smooth_nodes(rng, 1, 2, f_nodes)
    ph *= 0.01                                     # keep the phase small so the SciPy (fp64) spline values are exact enough
    tf = _unit_tf(rng, 1, 2)
    W = rng.uniform(0.5, 2.0, n_f)
    d = rng.standard_normal((2, n_f, 2))
    o = orc.full_batch(f_nodes, amp, ph, tf, None, k_min, df, d, W)
    mpmath.mp.dps = 40
    dh = hh = dd = mpmath.mpf(0)
    for c in range(2):
        for i in range(n_f):
            h = mpmath.mpc(0)
            for m in range(2):
                A = mpmath.mpf(float(CubicSpline(f_nodes, amp[0, m], bc_type="natural")(f[i])))
                P = mpmath.mpf(float(CubicSpline(f_nodes, ph[0, m], bc_type="natural")(f[i])))
                h += mpmath.mpc(*map(float, tf[0, m, c])) * A * mpmath.expj(-P)
            dc = mpmath.mpc(*map(float, d[c, i]))
            dh += mpmath.mpf(float(W[i])) * (mpmath.conj(dc) * h).real
            hh += mpmath.mpf(float(W[i])) * abs(h) ** 2
            dd += mpmath.mpf(float(W[i])) * abs(dc) ** 2
    assert o["d_h"][0] == pytest.approx(float(dh), rel=1e-12, abs=1e-12)
    assert o["h_h"][0] == pytest.approx(float(hh), rel=1e-12)
    assert o["logL"][0] == pytest.approx(float(dh - hh / 2 - dd / 2), rel=1e-12)


def test_interval_lookup_on_node_and_empty_intervals(orc):
    """R21: a bin that lands exactly on a node; intervals narrower than a bin (cfg-0 has 47 of them)."""
    k_min, df, n_f = 8, 1.0 / 64.0, 20
    f = np.arange(k_min, k_min + n_f) * df
    f_nodes = np.array([f[0], f[0] + 0.2 * df, f[0] + 0.3 * df, f[3], f[3] + 0.5 * df, f[10], f[-1]])
    rng = np.random.default_rng(3)
    amp, ph = _rand_smooth_nodes(rng, 2, 1, f_nodes)
    tf = _unit_tf(rng, 2, 1)
    W, d = rng.uniform(0.5, 2, n_f), rng.standard_normal((2, n_f, 2))
    o = orc.full_batch(f_nodes, amp, ph, tf, None, k_min, df, d, W)
    b = _brute_full(f_nodes, amp, ph, tf, None, k_min, df, d, W)
    np.testing.assert_allclose(o["logL"], b["logL"], rtol=1e-11)


# --------------------------------------------------------------------------- heterodyne (Eq. 10-19)
@pytest.fixture(scope="module")
def het_small(orc):
    """cfg-1 recipe on a 2^17 s grid (3.3k bins inside the band), 24 bins, 32 walkers."""
    wl = wlm.make_workload(1, n_w=32, t_obs=2.0 ** 17, n_knots=24)
    g = wl.grid
    f = g.freqs()
    lo, hi = f[0], f[-1]
    direct = lambda p, ff: orc.standin_direct(p, wl.modes_m, wl.c_lm, wl.kappa, ff, lo, hi)
    h1 = direct(wl.inj, f)
    wl.finish_distance(orc.inner(h1, h1, wl.W).real)
    h0 = direct(wl.inj, f)
    d = wl.make_data(h0)
    h0e = direct(wl.inj, wl.f_edges)
    summ = orc.het_prepare(g.k_min, g.df, d, wl.W, h0, wl.f_edges)
    return wl, f, d, h0, h0e, summ, direct


def _band_mask(f, e):
    return (f >= e[0]) & (f <= e[-1])


def test_summary_data_partition_exactness(orc, het_small):
    """sum_b A0(b) = sum_k W d conj(h0) and sum_b B0(b) = <h0|h0> over the het band; A1, B1 vs numpy."""
    wl, f, d, h0, h0e, s, _ = het_small
    m = _band_mask(f, wl.f_edges)
    dc, hc, W = _c(d), _c(h0), wl.W
    np.testing.assert_allclose(_c(s["A0"]).sum(axis=1), (W * dc * np.conj(hc))[:, m].sum(axis=1), rtol=1e-12)
    np.testing.assert_allclose(s["B0"].sum(), (W * np.abs(hc) ** 2)[:, m].sum(), rtol=1e-12)
    assert s["dd_band"] == pytest.approx((W * np.abs(dc) ** 2)[:, m].sum(), rel=1e-12)
    e = wl.f_edges
    idx = np.clip(np.searchsorted(e, f, side="right") - 1, 0, len(e) - 2)     # half-open bins, last closed (R13)
    fb = 0.5 * (e[:-1] + e[1:])
    for b in (0, 5, len(e) - 2):
        sel = m & (idx == b)
        assert sel.sum() > 0
        t = f[sel] - fb[b]
        np.testing.assert_allclose(_c(s["A1"])[:, b], (W[sel] * dc[:, sel] * np.conj(hc[:, sel]) * t).sum(axis=1),
                                   rtol=1e-10, atol=1e-12 * np.abs(_c(s["A0"])[:, b]).max())
        np.testing.assert_allclose(s["B1"][:, b], (W[sel] * np.abs(hc[:, sel]) ** 2 * t).sum(axis=1), rtol=1e-10,
                                   atol=1e-12 * s["B0"][:, b].max() * (e[b + 1] - e[b]))


def test_het_equals_full_at_reference(orc, het_small):
    """north_star invariant: h = h0 => r = 1 => het log L = -1/2 <d-h0|d-h0>_band to rounding."""
    wl, f, d, h0, h0e, s, _ = het_small
    amp, ph, tf, _ = orc.standin_nodes(wl.inj[None], wl.modes_m, wl.c_lm, wl.kappa, wl.f_edges, f[0], f[-1])
    r = orc.het_batch(wl.f_edges, amp, ph, tf, h0e, s)
    m = _band_mask(f, wl.f_edges)
    res = _c(d)[:, m] - _c(h0)[:, m]
    direct = -0.5 * (wl.W[m] * np.abs(res) ** 2).sum()
    assert r["logL"][0] == pytest.approx(direct, rel=1e-10)
    assert r["h_h"][0] == pytest.approx(s["B0"].sum(), rel=1e-13)
    assert r["d_h"][0] == pytest.approx(_c(s["A0"]).sum().real, rel=1e-13)


def test_het_exact_for_linear_ratio_and_known_deficit(orc, het_small):
    """h = (alpha + beta f) h0 => r exactly linear: Z[d,h] equals the dense <d|h>_band to rounding (Eq. 10-16),
    and Z[h,h] falls short of the dense <h|h>_band by exactly sum |r1|^2 B2 (the O(f^2) term Eq. 17 drops)."""
    wl, f, d, h0, h0e, s, _ = het_small
    alpha, beta = 0.8 - 0.3j, (25.0 + 40.0j)
    e = wl.f_edges
    he = (alpha + beta * e)[None, :] * _c(h0e)                     # template at the edges, per channel
    # feed it through the array entry: one "mode" per channel is not possible, so use tf = 1 and two calls
    m = _band_mask(f, e)
    hd = (alpha + beta * f)[None, :] * _c(h0)
    dense_dh = (wl.W[m] * (np.conj(_c(d)[:, m]) * hd[:, m]).real).sum(axis=1)
    dense_hh = (wl.W[m] * np.abs(hd[:, m]) ** 2).sum(axis=1)
    for c in range(2):
        amp = np.abs(he[c])[None, None, :]
        ph = -np.unwrap(np.angle(he[c]))[None, None, :]            # h = A e^{-i Psi}  (Eq. 7, R6)
        tf = np.zeros((1, 1, 2, 2)); tf[0, 0, c, 0] = 1.0
        h0e_c = h0e.copy()
        r = orc.het_batch(e, amp, ph, tf, h0e_c, s)
        r1 = beta
        deficit = abs(r1) ** 2 * s["B2"][c].sum()
        # the other channel contributes h = 0 => r = 0 => nothing
        assert r["d_h"][0] == pytest.approx(dense_dh[c], rel=1e-10)
        assert r["h_h"][0] == pytest.approx(dense_hh[c] - deficit, rel=1e-10)
        assert deficit / dense_hh[c] > 1e-9                        # the dropped term is visible, not rounding


def test_het_brute_force_tiny(orc):
    """2-4 bins x a few dozen dense points, everything random, numpy restatement of Eq. 11-19."""
    rng = np.random.default_rng(11)
    for n_b, n_f, n_m in ((2, 16, 1), (4, 40, 2), (3, 25, 3)):
        k_min, df = 10, 1.0 / 1024.0
        f = np.arange(k_min, k_min + n_f) * df
        e = np.sort(np.concatenate([[f[1] - 0.3 * df, f[-2] + 0.1 * df], rng.uniform(f[3], f[-4], n_b - 1)]))
        d, h0 = rng.standard_normal((2, n_f, 2)), rng.standard_normal((2, n_f, 2)) + 2.0
        W = rng.uniform(0.5, 2.0, n_f)
        h0e = rng.standard_normal((2, n_b + 1, 2)) + 2.0
        s = orc.het_prepare(k_min, df, d, W, h0, e)
        n_w = 3
        amp = rng.uniform(0.5, 2.0, (n_w, n_m, n_b + 1))
        ph = rng.uniform(-20, 20, (n_w, n_m, n_b + 1))
        tf = _unit_tf(rng, n_w, n_m)
        o = orc.het_batch(e, amp, ph, tf, h0e, s)
        # numpy restatement
        dc, hc = _c(d), _c(h0)
        idx = np.searchsorted(e, f, side="right") - 1
        idx[f == e[-1]] = n_b - 1
        inside = (f >= e[0]) & (f <= e[-1])
        fb = 0.5 * (e[:-1] + e[1:])
        A0 = np.zeros((2, n_b), complex); A1 = A0.copy(); B0 = np.zeros((2, n_b)); B1 = B0.copy()
        for i in np.nonzero(inside)[0]:
            b = idx[i]
            A0[:, b] += W[i] * dc[:, i] * np.conj(hc[:, i]); A1[:, b] += W[i] * dc[:, i] * np.conj(hc[:, i]) * (f[i] - fb[b])
            B0[:, b] += W[i] * abs(hc[:, i]) ** 2; B1[:, b] += W[i] * abs(hc[:, i]) ** 2 * (f[i] - fb[b])
        np.testing.assert_allclose(_c(s["A0"]), A0, rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(s["B1"], B1, rtol=1e-10, atol=1e-13)
        ddb = (W[inside] * np.abs(dc[:, inside]) ** 2).sum()
        for w in range(n_w):
            h = np.einsum("mc,me->ce", _c(tf[w]), amp[w] * np.exp(-1j * ph[w]))
            r = h / _c(h0e)
            r0, r1 = 0.5 * (r[:, :-1] + r[:, 1:]), (r[:, 1:] - r[:, :-1]) / np.diff(e)
            dh = (A0 * np.conj(r0) + A1 * np.conj(r1)).real.sum()
            hh = (B0 * np.abs(r0) ** 2 + 2 * B1 * (r0 * np.conj(r1)).real).sum()
            assert o["d_h"][w] == pytest.approx(dh, rel=1e-11, abs=1e-11)
            assert o["h_h"][w] == pytest.approx(hh, rel=1e-11)
            assert o["logL"][w] == pytest.approx(dh - hh / 2 - ddb / 2, rel=1e-11)


def test_het_reference_zero_is_an_error(orc, het_small):
    wl, f, d, h0, h0e, s, _ = het_small
    bad = h0e.copy(); bad[1, 3] = 0.0
    amp, ph, tf, _ = orc.standin_nodes(wl.inj[None], wl.modes_m, wl.c_lm, wl.kappa, wl.f_edges, f[0], f[-1])
    with pytest.raises(RuntimeError, match="-6"):
        orc.het_batch(wl.f_edges, amp, ph, tf, bad, s)


def test_het_tracks_dense_likelihood_near_reference(orc, het_small):
    """the brute-force likelihood verifies the heterodyned one.  Accuracy of the METHOD
    (not parity): for the 1e-3 Gaussian ball (|log L| of a few 1e3 at SNR 500) the heterodyned value tracks the
    dense one to < 1 % with only 24 bins (measured 0.2-0.6 %; 1e-4 with 128 bins)."""
    wl, f, d, h0, h0e, s, direct = het_small
    r = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, wl.f_edges, h0e, s)
    m = _band_mask(f, wl.f_edges)
    for w in range(8):
        h = _c(direct(wl.params[w], f))
        dense = -0.5 * (wl.W[m] * np.abs(_c(d)[:, m] - h[:, m]) ** 2).sum()
        assert abs(dense - r["logL"][w]) < 0.01 * abs(dense)
        assert dense < -100.0                                       # the ball really is off the peak


# --------------------------------------------------------------------------- noise normalisation
def test_noise_normalisation_statistic(orc):
    """<n n'> = S_n delta / 2  =>  (d_h - h_h)/sqrt(h_h) at Theta_true is N(0,1) over noise seeds (R16)."""
    wl = wlm.make_workload(1, n_w=1, t_obs=2.0 ** 15, n_knots=8)
    g = wl.grid
    f = g.freqs()
    h = orc.standin_direct(wl.inj, wl.modes_m, wl.c_lm, wl.kappa, f, f[0], f[-1])
    hh = orc.inner(h, h, wl.W).real
    z = []
    for s in range(200):
        n = wlm._draw_noise(90000 + s, g, 2)
        z.append(orc.inner(n, h, wl.W).real / math.sqrt(hh))
    z = np.array(z)
    assert abs(z.mean()) < 0.2
    assert 0.7 < z.var() < 1.4
    # E<n|n> = 2 n_f per channel
    nn = np.mean([orc.dd(wlm._draw_noise(91000 + s, g, 2), wl.W) for s in range(20)])
    assert nn == pytest.approx(4.0 * g.n_f, rel=0.05)


# ------------------------------------------- frequency-dependent transfer function (Eq. 8-9), SURVEY §8(f) item 1
def _rand_tf_nodes(rng, n_w, n_m, n_c, f_nodes):
    """smooth complex T^c_m at the nodes: (a + b x + c sin(2x + p)) e^{i(q + r x)}, x = normalised log f"""
    x = np.log(f_nodes / f_nodes[0]) / np.log(f_nodes[-1] / f_nodes[0])
    t = np.empty((n_w, n_m, n_c, len(f_nodes), 2))
    for idx in np.ndindex(n_w, n_m, n_c):
        a = rng.uniform(-1.0, 1.0, 6)
        mod = 1.0 + 0.3 * a[0] * x + 0.2 * a[1] * np.sin(2 * x + a[2])
        ang = 3.0 * a[3] + 2.0 * a[4] * x
        t[idx][:, 0], t[idx][:, 1] = mod * np.cos(ang), mod * np.sin(ang)
    return t


def test_tf_path_reduces_to_constant_tf_path(orc):
    """T constant over the nodes: its spline is that constant, so the result is orc_full_batch's (pinned above).
    Fails on a wrong Re/Im slot, a channel/mode index swap or a conjugation in the new path."""
    rng = np.random.default_rng(41)
    k_min, df, n_f, n_w, n_m = 7, 1.0 / 2048.0, 90, 4, 3
    f_lo, f_hi = k_min * df, (k_min + n_f - 1) * df
    f_nodes = wlm.geomspace_exact(f_lo * 0.95, f_hi * 1.02, 12)
    amp, ph = _rand_smooth_nodes(rng, n_w, n_m, f_nodes)
    tf = _unit_tf(rng, n_w, n_m) * rng.uniform(0.5, 1.5, (n_w, n_m, 2, 1))
    tfn = np.repeat(tf[:, :, :, None, :], len(f_nodes), axis=3)
    W = rng.uniform(0.5, 2.0, n_f)
    d = rng.standard_normal((2, n_f, 2))
    band = np.array([[f_lo, f_hi], [f_lo + 2.5 * df, f_hi - 7.1 * df], [f_lo, f_lo + 20 * df], [f_hi * 2, f_hi * 3]])
    a = orc.full_batch(f_nodes, amp, ph, tf, band, k_min, df, d, W)
    b = orc.full_batch_tf(f_nodes, amp, ph, tfn, band, k_min, df, d, W)
    for k in ("logL", "d_h", "h_h", "logL_direct"):
        np.testing.assert_allclose(b[k], a[k], rtol=1e-14, atol=1e-13)


def test_tf_path_linear_T_against_direct_numpy(orc):
    """Re T and Im T linear in f are reproduced exactly by any cubic spline, so the dense template must equal
    (alpha + beta f) x (the constant-T template with T = 1) bin by bin, computed here in numpy.
    Fails if T is evaluated at the wrong frequency / interval or multiplied in the wrong order."""
    rng = np.random.default_rng(43)
    k_min, df, n_f, n_m = 11, 1.0 / 1024.0, 70, 2
    f = np.arange(k_min, k_min + n_f) * df
    f_nodes = wlm.geomspace_exact(f[0] * 0.9, f[-1] * 1.1, 9)
    amp, ph = _rand_smooth_nodes(rng, 1, n_m, f_nodes)
    W = rng.uniform(0.5, 2.0, n_f)
    d = rng.standard_normal((2, n_f, 2))
    alpha = rng.standard_normal((n_m, 2)) + 1j * rng.standard_normal((n_m, 2))
    beta = (rng.standard_normal((n_m, 2)) + 1j * rng.standard_normal((n_m, 2))) / f[-1]
    tfn = np.empty((1, n_m, 2, len(f_nodes), 2))
    h_expect = np.zeros((2, n_f), dtype=complex)
    for m in range(n_m):
        one = np.zeros((1, 1, 2, 2)); one[..., 0] = 1.0
        hm = orc.full_batch(f_nodes, amp[:, m:m + 1], ph[:, m:m + 1], one, None, k_min, df, None, W, want_template=True)["h"]
        hm = hm[..., 0] + 1j * hm[..., 1]                          # [n_c][n_f], identical channels (T = 1)
        for c in range(2):
            tn = alpha[m, c] + beta[m, c] * f_nodes
            tfn[0, m, c, :, 0], tfn[0, m, c, :, 1] = tn.real, tn.imag
            h_expect[c] += (alpha[m, c] + beta[m, c] * f) * hm[c]
    o = orc.full_batch_tf(f_nodes, amp, ph, tfn, None, k_min, df, d, W, want_template=True)
    h = o["h"][..., 0] + 1j * o["h"][..., 1]
    np.testing.assert_allclose(h, h_expect, rtol=1e-12, atol=1e-30)
    dc = d[..., 0] + 1j * d[..., 1]
    assert o["d_h"][0] == pytest.approx(float(np.sum(W * (np.conj(dc) * h_expect).real)), rel=1e-11)
    assert o["h_h"][0] == pytest.approx(float(np.sum(W * np.abs(h_expect) ** 2)), rel=1e-12)


def test_tf_path_brute_force_scipy(orc):
    """tiny case, every spline by SciPy, sums by numpy complex arithmetic"""
    rng = np.random.default_rng(47)
    k_min, df, n_f, n_w, n_m = 4, 1.0 / 512.0, 40, 3, 2
    f = np.arange(k_min, k_min + n_f) * df
    f_nodes = wlm.geomspace_exact(f[0], f[-1], 7)
    amp, ph = _rand_smooth_nodes(rng, n_w, n_m, f_nodes)
    tfn = _rand_tf_nodes(rng, n_w, n_m, 2, f_nodes)
    W = rng.uniform(0.5, 2.0, n_f)
    d = rng.standard_normal((2, n_f, 2))
    dc = d[..., 0] + 1j * d[..., 1]
    band = np.array([[f[0], f[-1]], [f[3] + 0.2 * df, f[-4] - 0.3 * df], [f[0], f[10]]])
    o = orc.full_batch_tf(f_nodes, amp, ph, tfn, band, k_min, df, d, W)
    sp = lambda y: CubicSpline(f_nodes, y, bc_type="natural")(f)
    for w in range(n_w):
        mask = (f >= band[w, 0]) & (f <= band[w, 1])
        h = np.zeros((2, n_f), dtype=complex)
        for m in range(n_m):
            z = sp(amp[w, m]) * np.exp(-1j * sp(ph[w, m]))
            for c in range(2):
                h[c] += (sp(tfn[w, m, c, :, 0]) + 1j * sp(tfn[w, m, c, :, 1])) * z
        h *= mask
        dh = float(np.sum(W * (np.conj(dc) * h).real)); hh = float(np.sum(W * np.abs(h) ** 2))
        assert o["d_h"][w] == pytest.approx(dh, rel=1e-10, abs=1e-10)
        assert o["h_h"][w] == pytest.approx(hh, rel=1e-10)
        assert o["logL"][w] == pytest.approx(dh - 0.5 * hh - 0.5 * orc.dd(d, W), rel=1e-10)
        assert o["logL_direct"][w] == pytest.approx(-0.5 * float(np.sum(W * np.abs(dc - h) ** 2)), rel=1e-10)


def test_tlm_nodes_matches_scipy_derivative_and_chirp_time(orc):
    """Eq. 8: t_lm = t_ref - (1/2pi) dphi/df.  (i) the spline derivative at every node equals SciPy's;
    (ii) for the stand-in phase, whose 2 pi f t_c term is inside phi, t_ref = 0 gives -(t_c - tau(f)) up to the
    spline's own error (interior nodes of a 256-node grid): fails on a sign, a 2 pi, or an off-by-one node."""
    rng = np.random.default_rng(53)
    f_nodes = wlm.geomspace_exact(1e-4, 5e-2, 40)
    _, ph = _rand_smooth_nodes(rng, 2, 3, f_nodes)
    t = orc.tlm_nodes(f_nodes, ph, 123.0)
    for w in range(2):
        for m in range(3):
            dy = CubicSpline(f_nodes, ph[w, m], bc_type="natural")(f_nodes, 1)
            np.testing.assert_allclose(t[w, m], 123.0 - dy / TWO_PI, rtol=1e-9, atol=1e-9 * np.abs(dy).max() / TWO_PI)
    p = _row(mc_msun=4e5, q=0.3, t_c=9.0e4)
    fn = wlm.geomspace_exact(1e-4, 5e-2, 256)
    _, php, _, _ = orc.standin_nodes(p[None], mode_m=[2], c_lm=[1.0], kappa=0.5, f=fn, f_grid_lo=0.0, f_grid_hi=1.0)
    tl = orc.tlm_nodes(fn, php, 0.0)[0, 0]
    tau = 5.0 / 256.0 * p[0] ** (-5.0 / 3.0) * (math.pi * fn) ** (-8.0 / 3.0)
    sl = slice(20, 236)
    np.testing.assert_allclose(tl[sl], -(p[2] - tau[sl]), rtol=2e-6, atol=0.1)   # seconds; values 1e3 .. 4e6


# --------------------------------------------------------------------------- reference update and audit
def test_reference_update_picks_best_and_places_edges(orc, het_small):
    """best walker = plain scan (ties -> lowest index, NaN/inf never win); edges = numpy geomspace with exact ends,
    stopping at min(f_last, f_ISCO) with f_ISCO from the textbook formula (reading R12)."""
    from oracle import reference_update as ru
    assert ru.best_walker([1.0, 3.0, 3.0, -1.0]) == 1
    assert ru.best_walker([np.nan, -5.0, np.inf, -7.0]) == 1
    assert ru.best_walker([np.nan, np.inf]) == -1
    wl, f, d, h0, h0e, s, _ = het_small
    p = wl.params[3]
    e = ru.reference_edges(p, f[0], f[-1], 25)
    eta = p[1] / (1 + p[1]) ** 2
    f_isco = 6.0 ** -1.5 / (math.pi * p[0] * eta ** -0.6)
    assert e[0] == f[0] and e[-1] == pytest.approx(min(f[-1], f_isco), rel=1e-14)
    np.testing.assert_allclose(np.diff(np.log(e)), np.log(e[-1] / e[0]) / 24, rtol=1e-10)
    with pytest.raises(ValueError):
        ru.reference_edges(np.r_[1e3, 1.0, p[2:]], f[0], f[-1], 25)      # f_ISCO ~ 3e-6 Hz, below the grid


def test_audit_is_zero_at_d_equals_h_and_matches_numpy(orc, het_small):
    """Noiseless d = h: direct residual form bitwise 0, three-term form |.| <= 1e-6; on noisy data the
    three-term audit equals numpy complex arithmetic on the masked band."""
    from oracle import reference_update as ru
    wl, f, d, h0, h0e, s, _ = het_small
    g = wl.grid
    a = ru.audit(wl.inj[None], wl.modes_m, wl.c_lm, wl.kappa, g.k_min, g.df, g.n_f, h0, wl.W, wl.f_edges)
    assert a["logL_direct"][0] == 0.0
    assert abs(a["logL"][0]) <= 1e-6
    b = ru.audit(wl.params[:3], wl.modes_m, wl.c_lm, wl.kappa, g.k_min, g.df, g.n_f, d, wl.W, wl.f_edges)
    m = _band_mask(f, wl.f_edges)
    for w in range(3):
        hc = _c(orc.standin_direct(wl.params[w], wl.modes_m, wl.c_lm, wl.kappa, f, f[0], f[-1]))[:, m]
        res = _c(d)[:, m] - hc
        assert b["logL"][w] == pytest.approx(-0.5 * (wl.W[m] * np.abs(res) ** 2).sum(), rel=1e-9)
        assert b["logL_direct"][w] == pytest.approx(b["logL"][w], rel=1e-9)
        assert b["h_h"][w] == pytest.approx((wl.W[m] * np.abs(hc) ** 2).sum(), rel=1e-12)


def test_reference_update_then_het_equals_audit_at_new_reference(orc, het_small):
    """After the update the best walker IS the reference: r = 1, so its heterodyned log L equals its brute-force
    log L over the new band to rounding (north_star invariant), and nearby walkers agree closely."""
    from oracle import reference_update as ru
    wl, f, d, h0, h0e, s, _ = het_small
    g = wl.grid
    old = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, wl.f_edges, h0e, s)
    up = ru.reference_update(wl.params, old["logL"], wl.modes_m, wl.c_lm, wl.kappa, g.k_min, g.df, g.n_f, d, wl.W, 25)
    assert up["best"] == int(np.argmax(old["logL"]))
    het = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, up["f_edges"], up["h0_edges"], up["summ"])
    aud = ru.audit(wl.params, wl.modes_m, wl.c_lm, wl.kappa, g.k_min, g.df, g.n_f, d, wl.W, up["f_edges"])
    b = up["best"]
    assert het["logL"][b] == pytest.approx(aud["logL"][b], rel=1e-10, abs=1e-8)
    assert het["h_h"][b] == pytest.approx(aud["h_h"][b], rel=1e-12)
    # the method's own accuracy with 24 bins on a 1e-3 ball (cf. test_het_tracks_dense_likelihood_near_reference)
    assert np.all(np.abs(het["logL"] - aud["logL"]) < 0.01 * np.abs(aud["logL"]) + 1e-6)


# --------------------------------------------------------------------------- sampler step
def test_stretch_z_is_inverse_cdf_of_g():
    """g(z) ~ 1/sqrt(z) on [1/a, a]: CDF F(z) = (sqrt(a z) - 1)/(a - 1), so z(u) = ((a-1)u + 1)^2/a (R25)."""
    from oracle import sampler as sm
    u = np.linspace(0.0, 1.0, 11, endpoint=False)
    for a in (2.0, 3.5):
        z = sm.stretch_z(u, a)
        np.testing.assert_allclose((np.sqrt(a * z) - 1.0) / (a - 1.0), u, atol=1e-15)
        assert z[0] == pytest.approx(1.0 / a) and np.all((z >= 1.0 / a) & (z < a))


def _gauss_loglike(prec):
    def f(rows):
        return -0.5 * np.einsum("ni,ij,nj->n", rows, prec, rows), {}
    return f


@pytest.mark.parametrize("beta", [1.0, 0.25])
def test_stretch_move_keeps_gaussian_target(beta):
    """Invariance of the target under the move: a d = 3 correlated Gaussian sampled at inverse temperature beta has
    covariance C/beta.  Dropping z^(d-1), or using z^d, shifts the variance by tens of per cent."""
    from oracle import sampler as sm
    rng = np.random.default_rng(5)
    C = np.array([[1.0, 0.6, 0.0], [0.6, 2.0, -0.3], [0.0, -0.3, 0.5]])
    ll = _gauss_loglike(np.linalg.inv(C))
    n_w, d = 64, 3
    x = rng.normal(size=(1, n_w, d))
    logL = ll(x[0])[0][None, :].copy()
    lo, hi = np.full(d, -np.inf), np.full(d, np.inf)
    keep = []
    for it in range(1500):
        for half in (0, 1):
            sm.stretch_half(x, logL, half, [beta], lo, hi, d, 2.0, rng.random((1, n_w // 2)), rng.random((1, n_w // 2)),
                            rng.random((1, n_w // 2)), ll)
        if it >= 300:
            keep.append(x[0].copy())
    s = np.concatenate(keep)
    np.testing.assert_allclose(logL[0], ll(x[0])[0], rtol=1e-12)          # bookkeeping of the stored log L
    np.testing.assert_allclose(s.mean(axis=0), 0.0, atol=0.06 / np.sqrt(beta))
    np.testing.assert_allclose(np.cov(s.T), C / beta, rtol=0.08, atol=0.05 / beta)


def test_stretch_move_respects_prior_box_and_frozen_coordinates():
    from oracle import sampler as sm
    rng = np.random.default_rng(6)
    ll = _gauss_loglike(np.eye(3))
    x = rng.uniform(-1, 1, size=(2, 16, 3))
    x[..., 2] = 0.7                                                        # frozen: identical in every walker
    logL = np.stack([ll(x[t])[0] for t in range(2)])
    lo, hi = np.array([-1.0, -1.0, -np.inf]), np.array([1.0, 1.0, np.inf])
    for it in range(50):
        for half in (0, 1):
            sm.stretch_half(x, logL, half, [1.0, 0.1], lo, hi, 2, 2.0, rng.random((2, 8)), rng.random((2, 8)),
                            rng.random((2, 8)), ll)
    assert np.all(x[..., 2] == 0.7) and np.all(np.abs(x[..., :2]) <= 1.0)


def test_temperature_swaps_textbook_cases():
    """Equal betas: ln u < 0 always, every pair swaps.  Two temperatures: probability min(1, e^{dbeta dL}) (R27)."""
    from oracle import sampler as sm
    x = np.arange(2 * 4 * 1, dtype=float).reshape(2, 4, 1)
    logL = np.array([[0.0, -1.0, -2.0, -3.0], [-5.0, -0.5, -2.0, 1.0]])
    x0, l0 = x.copy(), logL.copy()
    done = sm.temperature_swaps(x, logL, [1.0, 1.0], np.full((1, 4), 0.999))
    assert done.all() and np.array_equal(x[0], x0[1]) and np.array_equal(logL[1], l0[0])
    x, logL = x0.copy(), l0.copy()
    # beta = (1, 0.5): ln q = (0.5 - 1)(L_cold - L_hot) = 0.5 (L_hot - L_cold) -> (-2.5, 0.25, 0, 2)
    u = np.exp(np.array([[-2.4, 0.1, -1e-9, 1.9]]))                         # just above / below each threshold
    u = np.minimum(u, 0.999999)
    done = sm.temperature_swaps(x, logL, [1.0, 0.5], u)
    assert done[0].tolist() == [False, True, True, True]
    # a three-rung sweep lets the best hot walker climb to the cold chain in one sweep
    x = np.array([[[0.0]], [[1.0]], [[2.0]]]); logL = np.array([[-9.0], [-5.0], [0.0]])
    sm.temperature_swaps(x, logL, [1.0, 0.5, 0.1], np.full((2, 1), 0.5))
    assert x[0, 0, 0] == 2.0 and logL[0, 0] == 0.0


def test_stopping_functions():
    """Module 1: extracted SNR against the limit.  Module 2: max log L unchanged (within 1) for 30
    consecutive checks."""
    from oracle import sampler as sm
    best, bi, snr = sm.population_stats([-3.0, np.nan, -1.0, -1.0], [3.0, 1.0, 8.0, 1.0], [1.0, 1.0, 4.0, 0.0])
    assert (best, bi, snr) == (-1.0, 2, 4.0)
    s1 = sm.StopSNR(20.0)
    assert not s1.check(19.9) and s1.check(20.0)
    s2 = sm.StopConverged(n_checks=3, tol=1.0)
    seq = [-10.0, -5.0, -4.5, -4.2, -3.9, -2.0, -1.9, -1.8, -1.7]
    assert [s2.check(v) for v in seq] == [False, False, False, False, False, False, False, False, True]


# --------------------------------------------------------------------------- per-walker node grids
def _pw_case(rng, n_w, n_m, n_nodes, n_f, k_min, df):
    f = (k_min + np.arange(n_f)) * df
    x = np.empty((n_w, n_nodes))
    for w in range(n_w):
        lo = f[0] * rng.uniform(0.8, 1.5)
        hi = f[-1] * rng.uniform(0.5, 1.1)
        x[w] = np.geomspace(lo, hi, n_nodes)
    xn = np.log(x / x[:, :1]) / np.log(x[:, -1:] / x[:, :1])
    amp = 1e-19 * (1.0 + rng.uniform(0.2, 1.0, (n_w, n_m, 1)) * xn[:, None, :] ** 2)
    ph = 40.0 * rng.uniform(-1, 1, (n_w, n_m, 1)) * xn[:, None, :] + 25.0 * np.cos(3 * xn[:, None, :] + rng.uniform(0, 6, (n_w, n_m, 1)))
    ang = rng.uniform(0, 2 * np.pi, (n_w, n_m, 2))
    tf = np.stack([np.cos(ang), np.sin(ang)], axis=-1)
    W = rng.uniform(0.5, 2.0, n_f) * 1e37
    d = rng.normal(size=(2, n_f, 2)) * 1e-19
    return f, x, amp, ph, tf, W, d


def test_per_walker_nodes_reduce_to_shared_nodes(orc):
    from oracle import per_walker as pw
    rng = np.random.default_rng(82)
    f, x, amp, ph, tf, W, d = _pw_case(rng, 5, 2, 12, 90, 40, 1e-5)
    x[:] = x[0]
    band = np.tile([[x[0, 0], x[0, -1]]], (5, 1))
    a = pw.full_batch_pw(x, amp, ph, tf, None, 40, 1e-5, d, W)
    b = orc.full_batch(x[0], amp, ph, tf, band, 40, 1e-5, d, W)
    for k in ("logL", "d_h", "h_h"):
        assert np.array_equal(a[k], b[k]), k


def test_per_walker_nodes_brute_force_scipy(orc):
    """different nodes per walker, zero outside each walker's own node span (R30): SciPy + numpy, one walker at a time"""
    from oracle import per_walker as pw
    rng = np.random.default_rng(83)
    f, x, amp, ph, tf, W, d = _pw_case(rng, 4, 2, 9, 70, 30, 2e-5)
    band = np.stack([x[:, 0] * 1.05, x[:, -1] * rng.uniform(0.7, 1.2, 4)], axis=1)
    for bnd in (None, band):
        got = pw.full_batch_pw(x, amp, ph, tf, bnd, 30, 2e-5, d, W)
        for w in range(4):
            b = np.array([[x[w, 0], x[w, -1]]]) if bnd is None else np.array([[max(x[w, 0], bnd[w, 0]), min(x[w, -1], bnd[w, 1])]])
            ref = _brute_full(x[w], amp[w:w + 1], ph[w:w + 1], tf[w:w + 1], b, 30, 2e-5, d, W)
            assert (f < x[w, 0]).any() or (f > x[w, -1]).any()                # some bins really are outside
            for k in ("logL", "d_h", "h_h"):
                assert got[k][w] == pytest.approx(ref[k][0], rel=1e-9, abs=1e-9 * abs(ref["logL"][0])), (k, w)


def test_per_walker_nodes_do_not_matter_for_a_spline_reproducible_template(orc):
    """Amplitude and phase linear in f are reproduced exactly by any natural spline, so two different node sets over
    the same span give the same likelihood."""
    from oracle import per_walker as pw
    rng = np.random.default_rng(84)
    n_f, k_min, df = 80, 25, 1e-5
    f = (k_min + np.arange(n_f)) * df
    xa = np.geomspace(f[3], f[-4], 7)
    xb = np.sort(np.r_[xa[0], rng.uniform(xa[0], xa[-1], 9), xa[-1]])
    W = rng.uniform(0.5, 2.0, n_f) * 1e37
    d = rng.normal(size=(2, n_f, 2)) * 1e-19
    tf = np.array([[[[0.6, 0.8], [1.0, 0.0]]]])
    lin = lambda x: (1e-19 * (1 + 300.0 * x)[None, None, :], (5.0 + 9e4 * x)[None, None, :])
    ra = pw.full_batch_pw(xa[None], *lin(xa), tf, None, k_min, df, d, W)
    rb = pw.full_batch_pw(xb[None], *lin(xb), tf, None, k_min, df, d, W)
    for k in ("logL", "d_h", "h_h"):
        assert ra[k][0] == pytest.approx(rb[k][0], rel=1e-11)


# --------------------------------------------------------------------------- not-a-knot boundary condition
@pytest.fixture
def notaknot(orc):
    orc.set_spline_bc(1)
    yield orc
    orc.set_spline_bc(0)


@pytest.mark.parametrize("n", [4, 5, 16, 257])
def test_notaknot_spline_matches_scipy(notaknot, n):
    """SciPy's CubicSpline default IS not-a-knot: values, second derivatives at the nodes."""
    orc = notaknot
    rng = np.random.default_rng(n)
    x = np.sort(rng.uniform(1e-4, 5e-2, n)) if n < 100 else np.geomspace(1e-4, 5e-2, n)
    y = np.cumsum(rng.normal(size=n)) * 50.0
    cs = CubicSpline(x, y)                                                       # bc_type='not-a-knot'
    q = np.r_[x, rng.uniform(x[0], x[-1], 300)]
    np.testing.assert_allclose(orc.spline_eval(x, y, q), cs(q), rtol=1e-10, atol=1e-9 * np.abs(y).max())
    M = orc.spline_second_derivatives(x, y)
    np.testing.assert_allclose(M, cs(x, 2), rtol=1e-7, atol=1e-8 * np.abs(cs(x, 2)).max())


def test_notaknot_reproduces_a_single_cubic_and_differs_from_natural(notaknot):
    """Not-a-knot reproduces any cubic exactly (natural does not: it forces y'' = 0 at the ends); the third
    derivative is continuous across x_1 and x_{n-2}; dense elimination of the full (n x n) system agrees."""
    orc = notaknot
    rng = np.random.default_rng(9)
    x = np.sort(rng.uniform(0.0, 2.0, 9))
    cub = lambda t: 1.0 - 2.0 * t + 0.7 * t ** 2 + 3.0 * t ** 3
    q = np.linspace(x[0], x[-1], 101)
    np.testing.assert_allclose(orc.spline_eval(x, cub(x), q), cub(q), rtol=1e-12)
    orc.set_spline_bc(0)
    assert np.max(np.abs(orc.spline_eval(x, cub(x), q) - cub(q))) > 1e-3
    orc.set_spline_bc(1)
    y = rng.normal(size=9)
    M = orc.spline_second_derivatives(x, y)
    h = np.diff(x)
    d3 = np.diff(M) / h
    assert d3[0] == pytest.approx(d3[1], rel=1e-9) and d3[-1] == pytest.approx(d3[-2], rel=1e-9)
    A = np.zeros((9, 9)); r = np.zeros(9)
    for j in range(1, 8):
        A[j, j - 1], A[j, j], A[j, j + 1] = h[j - 1] / 6, (h[j - 1] + h[j]) / 3, h[j] / 6
        r[j] = (y[j + 1] - y[j]) / h[j] - (y[j] - y[j - 1]) / h[j - 1]
    A[0, :3] = [-1 / h[0], 1 / h[0] + 1 / h[1], -1 / h[1]]
    A[8, -3:] = [-1 / h[-2], 1 / h[-2] + 1 / h[-1], -1 / h[-1]]
    np.testing.assert_allclose(M, np.linalg.solve(A, r), rtol=1e-9, atol=1e-10 * np.abs(M).max())


def test_notaknot_full_path_brute_force(notaknot):
    """the full-grid path under the switch against SciPy's not-a-knot spline + numpy complex sums"""
    orc = notaknot
    rng = np.random.default_rng(10)
    n_w, n_m, n_nodes, n_f, k_min, df = 3, 2, 8, 48, 20, 1e-4
    f = (k_min + np.arange(n_f)) * df
    x = np.geomspace(f[0] * 0.9, f[-1] * 1.1, n_nodes)
    amp = 1e-19 * rng.uniform(0.5, 2.0, (n_w, n_m, n_nodes))
    ph = np.cumsum(rng.uniform(0.0, 3.0, (n_w, n_m, n_nodes)), axis=2)
    ang = rng.uniform(0, 2 * np.pi, (n_w, n_m, 2))
    tf = np.stack([np.cos(ang), np.sin(ang)], axis=-1)
    W = rng.uniform(0.5, 2.0, n_f) * 1e37
    d = rng.normal(size=(2, n_f, 2)) * 1e-19
    got = orc.full_batch(x, amp, ph, tf, None, k_min, df, d, W)
    dc = d[..., 0] + 1j * d[..., 1]
    for w in range(n_w):
        h = np.zeros((2, n_f), complex)
        for m in range(n_m):
            hm = CubicSpline(x, amp[w, m])(f) * np.exp(-1j * CubicSpline(x, ph[w, m])(f))
            for c in range(2):
                h[c] += (tf[w, m, c, 0] + 1j * tf[w, m, c, 1]) * hm
        d_h = (W * (np.conj(dc) * h).real).sum()
        h_h = (W * np.abs(h) ** 2).sum()
        assert got["d_h"][w] == pytest.approx(d_h, rel=1e-9, abs=1e-9 * h_h)
        assert got["h_h"][w] == pytest.approx(h_h, rel=1e-10)


def test_counter_based_uniforms_are_splitmix64():
    """Known answers of SplitMix64 (seed 1234567: the reference implementation's first outputs), range, and the plain
    statistics of a uniform: mean 1/2, variance 1/12, no correlation between neighbouring streams or indices."""
    from oracle import sampler as sm
    kat = [6457827717110365317, 3203168211198807973, 9817491932198370423, 4593380528125082431, 16408922859458223821]
    assert [sm._mix(1234567 + sm._G * (i + 1)) for i in range(5)] == kat
    u = np.concatenate([sm.uniforms(99, it, kind, 500) for it in range(4) for kind in range(7)])
    assert u.min() >= 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.01 and abs(u.var() - 1.0 / 12.0) < 0.003
    a, b = sm.uniforms(99, 0, 0, 4000), sm.uniforms(99, 0, 1, 4000)
    assert abs(np.corrcoef(a, b)[0, 1]) < 0.05 and abs(np.corrcoef(a[:-1], a[1:])[0, 1]) < 0.05
    assert not np.array_equal(sm.uniforms(99, 1, 0, 8), sm.uniforms(99, 0, 0, 8))
    assert np.array_equal(sm.uniforms(99, 3, 2, 8), sm.uniforms(99, 3, 2, 8))        # a pure function of its counter


def test_sampler_run_keeps_gaussian_target():
    """the whole loop (halves + swaps, counter-based uniforms) on a 2-d Gaussian: cold chain keeps the target"""
    from oracle import sampler as sm
    C = np.array([[1.0, 0.5], [0.5, 2.0]])
    ll = _gauss_loglike(np.linalg.inv(C))
    rng = np.random.default_rng(3)
    x = rng.normal(size=(3, 32, 2))
    logL = np.stack([ll(x[t])[0] for t in range(3)])
    betas = np.array([1.0, 0.5, 0.1])
    keep = []
    for blk in range(40):
        n_acc = sm.run(x, logL, betas, np.full(2, -np.inf), np.full(2, np.inf), 2, 2.0, 7, 25 * blk, 25, ll)
        if blk >= 8:
            keep.append(x[0].copy())
        assert np.all(n_acc > 0)
    s = np.concatenate(keep)
    np.testing.assert_allclose(np.cov(s.T), C, rtol=0.2, atol=0.15)
    np.testing.assert_allclose(logL[0], ll(x[0])[0], rtol=1e-12)


# ------------------------------------------- three channels, per-channel weights (Eq. 3)
def _brute_full_wc(f_nodes, amp, phase, tf, band, k_min, df, d, Wc, t_shift=None):
    """_brute_full with one weight row per channel and an optional linear phase term outside the spline: SciPy natural
    spline + numpy complex arithmetic + math.fsum, the sums taken channel by channel."""
    n_w, n_m, _ = amp.shape
    n_c, n_f = Wc.shape
    f = np.arange(k_min, k_min + n_f, dtype=np.float64) * df
    dc = d[..., 0] + 1j * d[..., 1]
    out = {k: np.zeros(n_w) for k in ("logL", "d_h", "h_h")}
    dd = math.fsum(math.fsum(Wc[c] * np.abs(dc[c]) ** 2) for c in range(n_c))
    for w in range(n_w):
        mask = np.ones(n_f, bool) if band is None else (f >= band[w, 0]) & (f <= band[w, 1])
        dh = hh = 0.0
        for c in range(n_c):
            h = np.zeros(n_f, complex)
            for m in range(n_m):
                A = CubicSpline(f_nodes, amp[w, m], bc_type="natural")(f)
                P = CubicSpline(f_nodes, phase[w, m], bc_type="natural")(f)
                if t_shift is not None:
                    P = P + TWO_PI * f * t_shift[w]
                h += (tf[w, m, c, 0] + 1j * tf[w, m, c, 1]) * A * np.exp(-1j * P)
            h[~mask] = 0.0
            dh += math.fsum(Wc[c] * (np.conj(dc[c]) * h).real)
            hh += math.fsum(Wc[c] * np.abs(h) ** 2)
        out["d_h"][w], out["h_h"][w], out["logL"][w] = dh, hh, dh - 0.5 * hh - 0.5 * dd
    return out


def _tiny_case(rng, n_w, n_m, n_c, n_nodes, n_f):
    k_min, df = 7, 1.0 / 512.0
    f = np.arange(k_min, k_min + n_f) * df
    f_nodes = np.sort(np.concatenate([[f[0] * 0.9, f[-1] * 1.1], rng.uniform(f[1], f[-2], n_nodes - 2)]))
    amp, ph = _rand_smooth_nodes(rng, n_w, n_m, f_nodes)
    tf = _unit_tf(rng, n_w, n_m, n_c)
    d = rng.standard_normal((n_c, n_f, 2))
    Wc = rng.uniform(0.5, 2.0, (n_c, n_f)) * np.array([1.0, 3.0, 0.2])[:n_c, None]     # three different "PSDs"
    band = np.stack([rng.uniform(f[0], f[n_f // 3], n_w), rng.uniform(f[n_f // 2], f[-1], n_w)], axis=1)
    return k_min, df, f, f_nodes, amp, ph, tf, d, np.ascontiguousarray(Wc), band


def test_three_channels_equal_rows_reduce_to_shared_weights(orc):
    """W [n_c][n_f] with equal rows is the shared-W problem: every entry point that takes weights returns the same numbers."""
    rng = np.random.default_rng(41)
    k_min, df, f, f_nodes, amp, ph, tf, d, Wc, band = _tiny_case(rng, 4, 2, 3, 7, 48)
    W1 = np.ascontiguousarray(Wc[1])
    W3 = np.ascontiguousarray(np.tile(W1, (3, 1)))
    a = orc.full_batch(f_nodes, amp, ph, tf, band, k_min, df, d, W1)
    b = orc.full_batch(f_nodes, amp, ph, tf, band, k_min, df, d, W3)
    for k in ("logL", "d_h", "h_h", "logL_direct"):
        assert np.array_equal(a[k], b[k]), k
    tfn = _rand_tf_nodes(rng, 4, 2, 3, f_nodes)
    a = orc.full_batch_tf(f_nodes, amp, ph, tfn, band, k_min, df, d, W1)
    b = orc.full_batch_tf(f_nodes, amp, ph, tfn, band, k_min, df, d, W3)
    for k in ("logL", "d_h", "h_h", "logL_direct"):
        assert np.array_equal(a[k], b[k]), k
    assert orc.dd(d, W1) == orc.dd(d, W3) and orc.inner(d, d[::-1].copy(), W1) == orc.inner(d, d[::-1].copy(), W3)
    h0 = rng.standard_normal((3, 48, 2)) + 2.0
    e = np.array([f[2] - 0.1 * df, f[20], f[40] + 0.2 * df])
    sa, sb = orc.het_prepare(k_min, df, d, W1, h0, e), orc.het_prepare(k_min, df, d, W3, h0, e)
    for k in ("A0", "A1", "B0", "B1", "B2"):
        assert np.array_equal(sa[k], sb[k]), k
    assert sa["dd_band"] == sb["dd_band"]


@pytest.mark.parametrize("n_m,n_nodes,n_f", [(1, 5, 24), (3, 8, 49)])
def test_three_channels_three_psds_brute_force(orc, n_m, n_nodes, n_f):
    """n_c = 3 with three different weight rows against SciPy + numpy, channel by channel (Eq. 3: 4 Re sum over A, E, T
    of int a* b / S^c_n); a swapped or shared weight row fails it (the rows differ by factors 3 and 15)."""
    rng = np.random.default_rng(300 + n_m)
    k_min, df, f, f_nodes, amp, ph, tf, d, Wc, band = _tiny_case(rng, 3, n_m, 3, n_nodes, n_f)
    o = orc.full_batch(f_nodes, amp, ph, tf, band, k_min, df, d, Wc)
    r = _brute_full_wc(f_nodes, amp, ph, tf, band, k_min, df, d, Wc)
    for k in ("logL", "d_h", "h_h"):
        np.testing.assert_allclose(o[k], r[k], rtol=1e-11, atol=1e-11, err_msg=k)
    np.testing.assert_allclose(o["logL_direct"], o["logL"], rtol=1e-11, atol=1e-10)
    # the likelihood is additive over channels: three one-channel problems, each with its own row
    parts = [orc.full_batch(f_nodes, amp, ph, np.ascontiguousarray(tf[:, :, c:c + 1]), band, k_min, df,
                            np.ascontiguousarray(d[c:c + 1]), np.ascontiguousarray(Wc[c])) for c in range(3)]
    for k in ("logL", "d_h", "h_h"):
        np.testing.assert_allclose(o[k], sum(p[k] for p in parts), rtol=1e-12, atol=1e-12, err_msg=k)
    # frequency-dependent transfer function, same three rows
    tfn = _rand_tf_nodes(rng, 3, n_m, 3, f_nodes)
    o = orc.full_batch_tf(f_nodes, amp, ph, tfn, band, k_min, df, d, Wc)
    dc = _c(d)
    for w in range(3):
        mask = (f >= band[w, 0]) & (f <= band[w, 1])
        dh = hh = 0.0
        for c in range(3):
            h = np.zeros(n_f, complex)
            for m in range(n_m):
                A = CubicSpline(f_nodes, amp[w, m], bc_type="natural")(f)
                P = CubicSpline(f_nodes, ph[w, m], bc_type="natural")(f)
                T = CubicSpline(f_nodes, tfn[w, m, c, :, 0], bc_type="natural")(f) + 1j * CubicSpline(
                    f_nodes, tfn[w, m, c, :, 1], bc_type="natural")(f)
                h += T * A * np.exp(-1j * P)
            h[~mask] = 0.0
            dh += (Wc[c] * (np.conj(dc[c]) * h).real).sum()
            hh += (Wc[c] * np.abs(h) ** 2).sum()
        assert o["d_h"][w] == pytest.approx(dh, rel=1e-11, abs=1e-11) and o["h_h"][w] == pytest.approx(hh, rel=1e-11)


def test_hh_closed_form_three_flat_psds(orc):
    """<h|h> = sum_c |T^c|^2 (6/(D^2 S_c)) (f_lo^{-4/3} - f_hi^{-4/3}) (+ the Euler-Maclaurin term of the trapezoid
    sum) for three channels under three different flat PSDs, directly and through the spline path."""
    S = np.array([3.0e-40, 1.1e-39, 4.0e-41])
    tmod = np.array([1.0, 0.7, 1.6])
    grid = wlm.make_grid(2.0 ** 17)
    f = grid.freqs()
    w = np.ones(grid.n_f)
    w[0] = w[-1] = 0.5
    Wc = np.ascontiguousarray(4.0 * grid.df * w[None, :] / S[:, None])
    ang = np.array([0.3, 2.0, -1.1])
    p = np.concatenate([_row(mc_msun=50.0, q=1.0, t_c=0.6 * 2.0 ** 17, inv_d=1.0)[:5],
                        np.stack([tmod * np.cos(ang), tmod * np.sin(ang)], axis=1).ravel()])
    h = orc.standin_direct(p, [2], [1.0], 0.5, f, f[0], f[-1])
    assert h.shape == (3, grid.n_f, 2)
    hh = orc.inner(h, h, Wc).real
    gp = lambda x: -7.0 / 3.0 * x ** (-10.0 / 3.0)
    per_unit = 3.0 * (f[0] ** (-4.0 / 3.0) - f[-1] ** (-4.0 / 3.0)) + 4.0 * grid.df ** 2 / 12.0 * (gp(f[-1]) - gp(f[0]))
    expect = (tmod ** 2 / S).sum() * per_unit
    assert hh == pytest.approx(expect, rel=5e-6)
    f_nodes = wlm.geomspace_exact(1e-4, 0.05, 256)
    r = orc.full_batch_standin([2], [1.0], 0.5, p[None], f_nodes, grid.k_min, grid.df, grid.n_f, None, Wc)
    assert r["h_h"][0] == pytest.approx(expect, rel=2e-4)
    # one channel at a time: each term of the sum separately (a row applied to the wrong channel changes these)
    for c in range(3):
        hc = np.zeros_like(h)
        hc[c] = h[c]
        assert orc.inner(hc, hc, Wc).real == pytest.approx(tmod[c] ** 2 / S[c] * per_unit, rel=5e-6)


def test_het_three_channels_three_psds(orc):
    """heterodyne with per-channel weights: partition exactness of A0, B0 channel by channel against numpy, and
    het = full at h = h0 (north_star invariant) with three different PSDs."""
    wl = wlm.make_workload(1, n_w=8, t_obs=2.0 ** 17, n_knots=24, n_c=3)
    g = wl.grid
    f = g.freqs()
    assert wl.W.shape == (3, g.n_f) and not np.allclose(wl.W[0], wl.W[2])
    direct = lambda p, ff: orc.standin_direct(p, wl.modes_m, wl.c_lm, wl.kappa, ff, f[0], f[-1])
    h1 = direct(wl.inj, f)
    wl.finish_distance(orc.inner(h1, h1, wl.W).real)
    h0 = direct(wl.inj, f)
    d = wl.make_data(h0)
    h0e = direct(wl.inj, wl.f_edges)
    s = orc.het_prepare(g.k_min, g.df, d, wl.W, h0, wl.f_edges)
    m = _band_mask(f, wl.f_edges)
    dc, hc = _c(d), _c(h0)
    np.testing.assert_allclose(_c(s["A0"]).sum(axis=1), (wl.W * dc * np.conj(hc))[:, m].sum(axis=1), rtol=1e-12)
    np.testing.assert_allclose(s["B0"].sum(axis=1), (wl.W * np.abs(hc) ** 2)[:, m].sum(axis=1), rtol=1e-12)
    assert s["dd_band"] == pytest.approx((wl.W * np.abs(dc) ** 2)[:, m].sum(), rel=1e-12)
    amp, ph, tf, _ = orc.standin_nodes(wl.inj[None], wl.modes_m, wl.c_lm, wl.kappa, wl.f_edges, f[0], f[-1])
    assert tf.shape == (1, 1, 3, 2)
    r = orc.het_batch(wl.f_edges, amp, ph, tf, h0e, s)
    direct_ll = -0.5 * (wl.W[:, m] * np.abs(dc[:, m] - hc[:, m]) ** 2).sum()
    assert r["logL"][0] == pytest.approx(direct_ll, rel=1e-10)
    # near the reference the heterodyned value tracks the dense three-channel likelihood (method accuracy)
    amp, ph, tf, _ = orc.standin_nodes(wl.params, wl.modes_m, wl.c_lm, wl.kappa, wl.f_edges, f[0], f[-1])
    het = orc.het_batch(wl.f_edges, amp, ph, tf, h0e, s)
    for w in range(3):
        hw = _c(direct(wl.params[w], f))
        dense = (wl.W[:, m] * (np.conj(dc[:, m]) * hw[:, m]).real).sum() - 0.5 * (wl.W[:, m] * np.abs(hw[:, m]) ** 2).sum() \
            - 0.5 * s["dd_band"]
        assert abs(het["logL"][w] - dense) < 0.05 * max(1.0, abs(dense - direct_ll))


# ------------------------------------------- linear phase term outside the spline (reading R32)
def test_t_shift_equals_splining_the_full_phase(orc):
    """A natural cubic spline reproduces a linear function exactly, so Psi = spline(phase) + 2 pi f t_shift is the same
    function as spline(phase + 2 pi f_j t_shift): the two calls agree to the rounding of the larger phase."""
    rng = np.random.default_rng(52)
    k_min, df, f, f_nodes, amp, ph, tf, d, Wc, band = _tiny_case(rng, 5, 2, 2, 9, 64)
    W = np.ascontiguousarray(Wc[0])
    t = rng.uniform(-3e3, 3e3, 5)
    ph_full = ph + TWO_PI * f_nodes[None, None, :] * t[:, None, None]
    a = orc.full_batch(f_nodes, amp, ph, tf, band, k_min, df, d, W, t_shift=t)
    b = orc.full_batch(f_nodes, amp, ph_full, tf, band, k_min, df, d, W)
    scale = np.abs(ph_full).max()
    assert scale > 1e3
    for k in ("d_h", "h_h", "logL"):
        np.testing.assert_allclose(a[k], b[k], rtol=0, atol=1e-15 * scale * np.abs(b["h_h"]).max() * 50, err_msg=k)
    assert np.abs(a["d_h"] - orc.full_batch(f_nodes, amp, ph, tf, band, k_min, df, d, W)["d_h"]).max() > 1e-3   # it does something
    # SciPy + numpy with the term added after the spline
    r = _brute_full_wc(f_nodes, amp, ph, tf, band, k_min, df, d, np.ascontiguousarray(np.tile(W, (2, 1))), t_shift=t)
    for k in ("logL", "d_h", "h_h"):
        np.testing.assert_allclose(a[k], r[k], rtol=1e-10, atol=1e-10, err_msg=k)
    # frequency-dependent-T path and per-walker nodes take the same term
    tfn = _rand_tf_nodes(rng, 5, 2, 2, f_nodes)
    a = orc.full_batch_tf(f_nodes, amp, ph, tfn, band, k_min, df, d, W, t_shift=t)
    b = orc.full_batch_tf(f_nodes, amp, ph_full, tfn, band, k_min, df, d, W)
    np.testing.assert_allclose(a["logL"], b["logL"], rtol=0, atol=1e-15 * scale * np.abs(b["h_h"]).max() * 50)
    from oracle import per_walker as pw
    xw = np.tile(f_nodes, (5, 1))
    a = pw.full_batch_pw(xw, amp, ph, tf, band, k_min, df, d, W, t_shift=t)
    b = orc.full_batch(f_nodes, amp, ph, tf, band, k_min, df, d, W, t_shift=t)
    np.testing.assert_allclose(a["logL"], b["logL"], rtol=1e-13)


def test_t_shift_standin_split_and_het(orc):
    """stand-in: node phase without 2 pi f t_c, plus t_shift = t_c, is the stand-in's phase (for every mode: the linear
    term of (m/2) Psi(2f/m) is 2 pi f t_c); heterodyne: phase_e + 2 pi f_e t_shift enters exactly like a phase."""
    wl = wlm.make_workload(3, n_w=6, t_obs=2.0 ** 16, n_knots=12)
    f_nodes = wlm.geomspace_exact(wlm.F_LO, wlm.F_HI, 40)
    g = wl.grid
    f = g.freqs()
    a_full, p_full, tf, band = orc.standin_nodes(wl.params, wl.modes_m, wl.c_lm, wl.kappa, f_nodes, f[0], f[-1])
    a_spl, p_spl, tf2, band2 = orc.standin_nodes(wl.params, wl.modes_m, wl.c_lm, wl.kappa, f_nodes, f[0], f[-1], split_tc=True)
    assert np.array_equal(a_full, a_spl) and np.array_equal(tf, tf2) and np.array_equal(band, band2)
    lin = TWO_PI * f_nodes[None, None, :] * wl.params[:, 2][:, None, None]
    np.testing.assert_allclose(p_spl + lin, p_full, rtol=0, atol=1e-15 * np.abs(p_full).max() * 4)
    assert np.all(np.abs(p_spl[..., -1]) < 0.01 * np.abs(p_full[..., -1]))   # at the top of the band almost nothing is left to spline
    rng = np.random.default_rng(8)
    d = rng.standard_normal((2, g.n_f, 2)) * 1e-19
    run = lambda split: orc.full_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, f_nodes, g.k_min, g.df, g.n_f, d,
                                               wl.W, split_tc=split)
    a, b = run(True), run(False)
    np.testing.assert_allclose(a["h_h"], b["h_h"], rtol=1e-9)
    np.testing.assert_allclose(a["d_h"], b["d_h"], rtol=0, atol=1e-9 * np.sqrt(np.abs(b["h_h"]).max() * orc.dd(d, wl.W)))
    # heterodyne array entry: t_shift against the same term added to the edge phases
    e = wl.f_edges
    h0 = rng.standard_normal((2, g.n_f, 2)) + 2.0
    h0e = rng.standard_normal((2, len(e), 2)) + 2.0
    s = orc.het_prepare(g.k_min, g.df, rng.standard_normal((2, g.n_f, 2)), rng.uniform(0.5, 2.0, g.n_f), h0, e)   # O(1) scales
    amp_e = rng.uniform(0.5, 2.0, (6, wl.n_m, len(e)))
    ph_e = rng.uniform(-20, 20, (6, wl.n_m, len(e)))
    t = rng.uniform(-50.0, 50.0, 6)
    a = orc.het_batch(e, amp_e, ph_e, tf, h0e, s, t_shift=t)
    b = orc.het_batch(e, amp_e, ph_e + TWO_PI * e[None, None, :] * t[:, None, None], tf, h0e, s)
    for k in ("logL", "d_h", "h_h"):
        np.testing.assert_allclose(a[k], b[k], rtol=1e-11, atol=1e-11 * np.abs(b["h_h"]).max(), err_msg=k)
    assert np.abs(a["d_h"] - orc.het_batch(e, amp_e, ph_e, tf, h0e, s)["d_h"]).max() > 1e-3 * np.abs(b["d_h"]).max()
