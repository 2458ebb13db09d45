"""Shared by the GPU parity tests: finish a seeded workload WITH THE ORACLE (so that every input both sides see
comes from oracle/ or from the seeded generator, never from the CUDA path) and small comparison utilities."""
import numpy as np

from paper_2111_01064_b200 import workloads as wlm


def tol_ll(ref):
    """BASELINE.json north_star: |delta log L| <= 1e-6 * max(1, |log L|) for FP64."""
    return 1e-6 * np.maximum(1.0, np.abs(ref))


def assert_close_ll(got, ref, what=""):
    got, ref = np.asarray(got, dtype=np.float64), np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape, (what, got.shape, ref.shape)
    err = np.abs(got - ref)
    bad = err > tol_ll(ref)
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} outside tolerance; worst |err|={err.max():.3e} " \
                          f"at {int(err.argmax())} (ref {ref[err.argmax()]:.6e})"


def dev(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")


def make_ctx(wl, precision=0):
    from paper_2111_01064_b200 import binding
    ctx = binding.Context(n_modes=wl.n_m, precision=precision, n_channels=wl.n_c)
    ctx.standin_config(wl.modes_l, wl.modes_m, wl.c_lm, wl.kappa)
    return ctx


def check_triplet(got, ref, what):
    """log L at the north_star bar; d_h and h_h separately at 1e-6 max(1, |h_h|) so that a cancelling pair cannot hide"""
    logL, d_h, h_h = (x.cpu().numpy() for x in got)
    assert_close_ll(logL, ref["logL"], what + " logL")
    scale = np.maximum(1.0, np.abs(ref["h_h"]))
    assert np.all(np.abs(d_h - ref["d_h"]) <= 1e-6 * np.maximum(scale, np.abs(ref["d_h"]))), what + " d_h"
    assert np.all(np.abs(h_h - ref["h_h"]) <= 1e-6 * scale), what + " h_h"


def oracle_setup_full(orc, wl: wlm.Workload):
    g = wl.grid
    run = lambda params, d, tmpl=False: orc.full_batch_standin(
        wl.modes_m, wl.c_lm, wl.kappa, params, wl.f_nodes, g.k_min, g.df, g.n_f, d, wl.W, want_template=tmpl)
    if not wl.finished:
        wl.finish_distance(run(wl.inj[None], None)["h_h"][0])
    h = run(wl.inj[None], None, True)["h"]
    d = wl.make_data(h)
    return d, run


def oracle_setup_het(orc, wl: wlm.Workload):
    g = wl.grid
    f = g.freqs()
    lo, hi = float(f[0]), float(f[-1])
    direct = lambda p, ff: orc.standin_direct(p, wl.modes_m, wl.c_lm, wl.kappa, ff, lo, hi)
    if not wl.finished:
        h1 = direct(wl.inj, f)
        wl.finish_distance(orc.inner(h1, h1, wl.W).real)
    h0 = direct(wl.inj, f)
    d = wl.make_data(h0)
    h0e = direct(wl.inj, wl.f_edges)
    summ = orc.het_prepare(g.k_min, g.df, d, wl.W, h0, wl.f_edges)
    return d, h0, h0e, summ


def rand_smooth_nodes(rng, n_w, n_m, f_nodes, phase_scale=200.0):
    """smooth random amplitude/phase node arrays (not the stand-in), for the array entry points"""
    x = np.log(f_nodes / f_nodes[0]) / np.log(f_nodes[-1] / f_nodes[0])
    amp = np.empty((n_w, n_m, len(f_nodes)))
    ph = np.empty((n_w, n_m, len(f_nodes)))
    for w in range(n_w):
        for m in range(n_m):
            a = rng.uniform(0.5, 2.0, 4)
            amp[w, m] = 1e-19 * (a[0] + a[1] * x + a[2] * np.sin(3 * x + a[3]))
            b = rng.uniform(-1.0, 1.0, 4)
            ph[w, m] = phase_scale * (b[0] + b[1] * x + b[2] * x ** 2 + np.cos(2 * x + b[3]))
    return amp, ph


def unit_tf(rng, n_w, n_m, n_c=2):
    ang = rng.uniform(0, 2 * np.pi, (n_w, n_m, n_c))
    return np.stack([np.cos(ang), np.sin(ang)], axis=-1)


def pw_case(rng, n_w, n_m, n_nodes, n_f, k_min, df):
    """per-walker node grids: log-spaced nodes over each walker's own span (some start above the grid's first bin,
    some end below its last), smooth amplitude / phase at the nodes, unit-modulus transfer factors, random data"""
    f = (k_min + np.arange(n_f)) * df
    x = np.empty((n_w, n_nodes))
    for w in range(n_w):
        x[w] = np.geomspace(f[0] * rng.uniform(0.8, 1.5), f[-1] * rng.uniform(0.4, 1.1), n_nodes)
    xn = np.log(x / x[:, :1]) / np.log(x[:, -1:] / x[:, :1])
    amp = 1e-19 * (1.0 + rng.uniform(0.2, 1.0, (n_w, n_m, 1)) * xn[:, None, :] ** 2)
    ph = 4000.0 * rng.uniform(-1, 1, (n_w, n_m, 1)) * xn[:, None, :] + 25.0 * np.cos(3 * xn[:, None, :] + rng.uniform(0, 6, (n_w, n_m, 1)))
    ang = rng.uniform(0, 2 * np.pi, (n_w, n_m, 2))
    tf = np.ascontiguousarray(np.stack([np.cos(ang), np.sin(ang)], axis=-1))
    W = rng.uniform(0.5, 2.0, n_f) * 1e37
    d = rng.normal(size=(2, n_f, 2)) * 1e-19
    return f, x, np.ascontiguousarray(amp), np.ascontiguousarray(ph), tf, W, d
