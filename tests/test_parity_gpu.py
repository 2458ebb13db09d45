"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI (binding.Context), against the CPU oracle on the
same seeded inputs.  Tolerance (BASELINE.json north_star): |delta log L| <= 1e-6 max(1, |log L|) in FP64; d_h and h_h
are held to the same bound separately (scaled by max(1, |h_h|)) so that a cancelling pair of errors cannot hide."""
import math

import numpy as np
import pytest

from paper_2111_01064_b200 import workloads as wlm
from helpers import (assert_close_ll, check_triplet, dev, make_ctx, oracle_setup_full, oracle_setup_het, rand_smooth_nodes,
                     tol_ll, unit_tf)

pytestmark = pytest.mark.gpu


# ------------------------------------------------------------------------------------------- full grid
@pytest.fixture(scope="module")
def cfg0(orc, torch_cuda):
    wl = wlm.make_workload(0)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    return wl, d, run, ctx


def test_cfg0_full_standin_parity(cfg0, torch_cuda):
    """BASELINE.json config 0 in full: 64 walkers, 256 nodes, 6540 bins, noiseless; log L[0] = 0."""
    wl, d, run, ctx = cfg0
    ref = run(wl.params, d)
    got = ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))
    check_triplet(got, ref, "cfg0")
    assert abs(float(got[0][0])) <= 1e-6
    assert math.sqrt(float(got[2][0])) == pytest.approx(500.0, rel=1e-9)


def test_dd_matches_oracle(cfg0, orc):
    wl, d, run, ctx = cfg0
    dd_full, _ = ctx.get_dd()
    ref = orc.dd(d, wl.W)
    assert abs(dd_full - ref) <= 1e-12 * abs(ref)


def test_cfg0_rerun_is_bit_identical(cfg0, torch_cuda):
    wl, d, run, ctx = cfg0
    p = dev(torch_cuda, wl.params)
    a = [x.clone() for x in ctx.full_batch_standin(wl.f_nodes, p)]
    b = ctx.full_batch_standin(wl.f_nodes, p)
    for x, y in zip(a, b):
        assert torch_cuda.equal(x, y)


@pytest.mark.parametrize("n_w", [1, 31, 33, 200])
def test_full_standin_ragged_batches(cfg0, torch_cuda, n_w):
    wl, d, run, ctx = cfg0
    rng = np.random.default_rng(n_w)
    idx = rng.integers(0, wl.n_w, n_w)
    params = wl.params[idx].copy()
    params[:, 0] *= rng.uniform(0.7, 1.4, n_w)          # new masses -> new bands
    ref = run(params, d)
    got = ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, params))
    check_triplet(got, ref, f"ragged n_w={n_w}")


def test_full_standin_empty_batch_is_noop(cfg0, torch_cuda):
    wl, d, run, ctx = cfg0
    got = ctx.full_batch_standin(wl.f_nodes, torch_cuda.empty((0, wl.P), dtype=torch_cuda.float64, device="cuda"))
    assert all(x.numel() == 0 for x in got)


def test_full_template_matches_oracle(cfg0, torch_cuda):
    """The dense template the fused kernel integrates (never stored on the hot path), written out by the utility."""
    wl, d, run, ctx = cfg0
    for w in (0, 5, 17):
        ref = run(wl.params[w][None], None, True)["h"]
        got = ctx.full_template_standin(wl.f_nodes, wl.params[w]).cpu().numpy()
        scale = np.abs(ref).max()
        assert np.abs(got - ref).max() <= 1e-9 * scale, w


def test_walker_outside_grid_gets_minus_half_dd(cfg0, torch_cuda):
    wl, d, run, ctx = cfg0
    rng = np.random.default_rng(3)
    f_nodes = wl.f_nodes
    amp, ph = rand_smooth_nodes(rng, 3, 1, f_nodes)
    tf = unit_tf(rng, 3, 1)
    band = np.array([[1.0, 2.0], [1e-9, 2e-9], [3e-3, 2e-3]])      # above, below, inverted
    logL, d_h, h_h = ctx.full_batch(f_nodes, dev(torch_cuda, amp), dev(torch_cuda, ph), dev(torch_cuda, tf), dev(torch_cuda, band))
    dd_full, _ = ctx.get_dd()
    assert np.all(d_h.cpu().numpy() == 0.0) and np.all(h_h.cpu().numpy() == 0.0)
    np.testing.assert_allclose(logL.cpu().numpy(), -0.5 * dd_full, rtol=1e-15)


@pytest.mark.parametrize("n_m,banded,n_w", [(1, False, 40), (1, True, 97), (3, True, 50), (6, False, 33)])
def test_full_arrays_entry_point(orc, torch_cuda, n_m, banded, n_w):
    """ll_full_batch with caller arrays (not the stand-in), several modes, per-walker bands, noisy data."""
    from paper_2111_01064_b200 import binding
    rng = np.random.default_rng(1000 + 10 * n_m + n_w)
    grid = wlm.make_grid(2.0 ** 16)
    f = grid.freqs()
    f_nodes = wlm.geomspace_exact(wlm.F_LO, wlm.F_HI, 61)
    W = wlm.trapezoid_weights(grid)
    amp, ph = rand_smooth_nodes(rng, n_w, n_m, f_nodes)
    tf = unit_tf(rng, n_w, n_m)
    sigma = np.sqrt(wlm.psd_sn(f) / (4 * grid.df))
    d = rng.standard_normal((2, grid.n_f, 2)) * sigma[None, :, None]
    band = None
    if banded:
        lo = rng.uniform(0.5e-4, 5e-3, n_w)
        band = np.stack([lo, lo * rng.uniform(1.0, 40.0, n_w)], axis=1)
        band[0] = [f[10], f[10]]            # a single bin
        band[1] = [f[0], f[-1]]             # exactly the whole grid
    ref = orc.full_batch(f_nodes, amp, ph, tf, band, grid.k_min, grid.df, d, W)
    ctx = binding.Context(n_modes=n_m)
    ctx.set_data(grid.n_f, grid.k_min, grid.df, dev(torch_cuda, d), dev(torch_cuda, W))
    got = ctx.full_batch(f_nodes, dev(torch_cuda, amp), dev(torch_cuda, ph), dev(torch_cuda, tf),
                         None if band is None else dev(torch_cuda, band))
    check_triplet(got, ref, f"arrays n_m={n_m}")
    ctx.destroy()


def test_full_multimode_standin(orc, torch_cuda):
    """six-mode stand-in through the full-grid path (generic-n_m kernel)."""
    wl = wlm.make_workload(3, n_w=48, t_obs=2.0 ** 16, n_knots=24)
    wl.path = "full"
    wl.f_nodes = wlm.geomspace_exact(wlm.F_LO, wlm.F_HI, 200)
    wl.params[:, 0] *= np.random.default_rng(5).uniform(0.5, 2.0, wl.n_w)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    ref = run(wl.params, d)
    got = ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))
    check_triplet(got, ref, "6-mode full")
    ctx.destroy()


def test_cfg2_scaled_multi_tile(orc, torch_cuda):
    """config-2 recipe at 1/16 of the grid (98k bins, 1024 nodes, noisy), 600 walkers: several walker blocks,
    many frequency tiles, ragged tails in both directions."""
    wl = wlm.make_workload(2, n_w=600, t_obs=31557600.0 / 16)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    ref = run(wl.params, d)
    got = ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))
    check_triplet(got, ref, "cfg2/16")
    pairs, _ = ctx.last_full_stats()
    # active pairs = sum over walkers of bins inside the band (reading R10), counted by the oracle's mask
    f = g.freqs()
    _, _, _, band = orc.standin_nodes(wl.params, wl.modes_m, wl.c_lm, wl.kappa, wl.f_nodes, f[0], f[-1])
    expect = sum(int(((f >= lo) & (f <= hi)).sum()) for lo, hi in band)
    assert pairs == expect
    ctx.destroy()


def test_cfg2_full_size_sampled(orc, torch_cuda):
    """BASELINE.json config 2 at full size in the launch configuration bench.py times (16384 walkers, 1024 nodes,
    1 574 725 bins, noisy); the oracle recomputes a sample of walkers one by one."""
    wl = wlm.make_workload(2)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))]
    fis = np.array([orc.standin_fisco(p) for p in wl.params])
    sample = sorted({0, int(fis.argmin()), int(fis.argmax()), 1, 4097, 16383} | set(range(37, 16384, 2048)))
    ref = run(wl.params[sample], d)
    check_triplet([__import__("torch").as_tensor(x[sample]) for x in got], ref, "cfg2 sampled")
    assert np.all(np.isfinite(got[0]))
    # properties that hold for every walker: Cauchy-Schwarz and log L <= max over 1/D
    dd_full, _ = ctx.get_dd()
    assert np.all(got[1] ** 2 <= dd_full * got[2] * (1 + 1e-9))
    np.testing.assert_allclose(got[0], got[1] - 0.5 * got[2] - 0.5 * dd_full, rtol=1e-13)
    # Module-1 sized batches of the same walkers on the same grid (80 walkers x 4 temperatures, half of
    # them per likelihood call) take the small-batch route (one-block sort and cost plan, block-per-system spline, one-warp
    # blocks over cost-balanced work items, k_finalize_small); every walker must come out as in the big batch, up to
    # summation order
    for n_small in (160, 37):
        sm = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params[:n_small]))]
        assert ctx.last_full_stats()[1] > 8 * 64 * (n_small // 32 + 1) // 2          # thousands of work items, not a handful of walker blocks
        for a, b in zip(sm, got):                          # other tiles -> other re-sync points of the recurrence
            assert np.all(np.abs(a - b[:n_small]) <= 1e-7 * np.maximum(1.0, np.abs(b[:n_small])))
    ctx.destroy()


# ------------------------------------------- full grid, frequency-dependent transfer function (Eq. 8-9)
def _smooth_tf_nodes(rng, n_w, n_m, f_nodes, n_c=2):
    """smooth complex T^c_m at the nodes (not a physical response: its formula is in the paper's ref. [44])"""
    x = np.log(f_nodes / f_nodes[0]) / np.log(f_nodes[-1] / f_nodes[0])
    a = rng.uniform(-1.0, 1.0, (n_w, n_m, n_c, 6, 1))
    mod = 1.0 + 0.3 * a[..., 0, :] * x + 0.2 * a[..., 1, :] * np.sin(2 * x + a[..., 2, :])
    ang = 3.0 * a[..., 3, :] + 2.0 * a[..., 4, :] * x
    return np.ascontiguousarray(np.stack([mod * np.cos(ang), mod * np.sin(ang)], axis=-1))


@pytest.mark.parametrize("n_m,banded,n_w", [(1, False, 40), (1, True, 97), (3, True, 50)])
def test_full_tf_entry_point(orc, torch_cuda, n_m, banded, n_w):
    """ll_full_batch_tf against the oracle: several walker blocks and tiles, ragged bands, 1 and 3 modes."""
    rng = np.random.default_rng(900 + n_m + n_w)
    grid = wlm.make_grid(2.0 ** 15)
    f = grid.freqs()
    f_nodes = wlm.geomspace_exact(wlm.F_LO, wlm.F_HI, 96)
    amp, ph = rand_smooth_nodes(rng, n_w, n_m, f_nodes)
    amp *= 1e19 * 0.05                                     # O(1) templates against O(1) data
    tfn = _smooth_tf_nodes(rng, n_w, n_m, f_nodes)
    W = rng.uniform(0.5, 2.0, grid.n_f)
    d = rng.standard_normal((2, grid.n_f, 2))
    band = None
    if banded:
        lo = rng.uniform(f[0], f[grid.n_f // 3], n_w)
        hi = rng.uniform(f[grid.n_f // 2], f[-1], n_w)
        band = np.stack([lo, hi], axis=1)
        band[0] = [f[-1] * 2, f[-1] * 3]                   # misses the grid
        band[1] = [f[5], f[5]]                             # a single bin
    ref = orc.full_batch_tf(f_nodes, amp, ph, tfn, band, grid.k_min, grid.df, d, W)
    from paper_2111_01064_b200 import binding
    ctx = binding.Context(n_modes=n_m)
    ctx.set_data(grid.n_f, grid.k_min, grid.df, dev(torch_cuda, d), dev(torch_cuda, W))
    got = ctx.full_batch_tf(f_nodes, dev(torch_cuda, amp), dev(torch_cuda, ph), dev(torch_cuda, tfn),
                            None if band is None else dev(torch_cuda, band))
    check_triplet(got, ref, f"tf n_m={n_m}")
    again = ctx.full_batch_tf(f_nodes, dev(torch_cuda, amp), dev(torch_cuda, ph), dev(torch_cuda, tfn),
                              None if band is None else dev(torch_cuda, band))
    assert all(torch_cuda.equal(a, b) for a, b in zip(got, again))
    # a transfer function that is constant over the nodes must give what ll_full_batch gives (same library)
    tf_const = np.ascontiguousarray(tfn[:, :, :, 0, :])
    tfn_c = np.ascontiguousarray(np.repeat(tf_const[:, :, :, None, :], len(f_nodes), axis=3))
    a = ctx.full_batch(f_nodes, dev(torch_cuda, amp), dev(torch_cuda, ph), dev(torch_cuda, tf_const),
                       None if band is None else dev(torch_cuda, band))
    b = ctx.full_batch_tf(f_nodes, dev(torch_cuda, amp), dev(torch_cuda, ph), dev(torch_cuda, tfn_c),
                          None if band is None else dev(torch_cuda, band))
    check_triplet(b, {k: v.cpu().numpy() for k, v in zip(("logL", "d_h", "h_h"), a)}, "tf const vs constant-T path")
    ctx.destroy()


def test_tlm_nodes_parity(orc, torch_cuda):
    """Eq. 8 utility against the oracle (spline derivative at the nodes)."""
    rng = np.random.default_rng(77)
    wl = wlm.make_workload(0)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    f = g.freqs()
    am, ph, _, o_bd = orc.standin_nodes(wl.params[:37], wl.modes_m, wl.c_lm, wl.kappa, wl.f_nodes, f[0], f[-1])
    # ll_standin_nodes: the library's own node arrays in the caller layout against the oracle's
    g_am, g_ph, g_bd = (x.cpu().numpy() for x in ctx.standin_nodes(wl.f_nodes, dev(torch_cuda, wl.params[:37]),
                                                                   with_band=True))
    np.testing.assert_allclose(g_bd, o_bd, rtol=1e-14)
    # absolute term: the taper's s = (1+kappa-x)/kappa cancels near its zero, where the amplitude itself is ~1e-12 of its peak
    np.testing.assert_allclose(g_am, am, rtol=1e-13, atol=1e-15 * am.max())
    np.testing.assert_allclose(g_ph, ph, rtol=1e-14, atol=1e-9)
    ref = orc.tlm_nodes(wl.f_nodes, ph, 1000.0)
    got = ctx.tlm_nodes(wl.f_nodes, dev(torch_cuda, ph), 1000.0).cpu().numpy()
    np.testing.assert_allclose(got, ref, rtol=1e-9, atol=1e-9 * np.abs(ref).max())
    ctx.destroy()


# ------------------------------------------------------------------ full grid, FP32-accumulate variant
MIXED_ABS_TOL = 1e-3  # BASELINE.json north_star: "<= 1e-3 absolute for any mixed-precision variant"


def check_mixed(got, ref, what, tol=MIXED_ABS_TOL):
    logL, d_h, h_h = (np.asarray(x.cpu().numpy() if hasattr(x, "cpu") else x) for x in got)
    for name, a, b in (("logL", logL, ref["logL"]), ("d_h", d_h, ref["d_h"])):
        err = np.abs(a - b)
        assert err.max() <= tol, f"{what} {name}: worst |err| {err.max():.3e} at {int(err.argmax())}"
    # <h|h> stays in FP64 in this variant (reading R15): FP64 bar
    assert np.all(np.abs(h_h - ref["h_h"]) <= 1e-6 * np.maximum(1.0, np.abs(ref["h_h"]))), what + " h_h"
    return float(np.abs(logL - ref["logL"]).max())


def test_cfg0_mixed_precision_parity(cfg0, torch_cuda):
    """FP32-accumulate variant (reading R15) on config 0: a logic / ragged-shape check, not a BASELINE case for
    this variant (config 2 is).  Noiseless SNR 500-1000 on only 6.5k bins makes the per-bin terms of <d|h> ~240x
    larger than config 2's; binary32 rounding is relative to each term, so the absolute error grows like
    <d|h>/sqrt(n_bins): 2^-24 * 1e6 / sqrt(3e3) * (a few roundings) ~ 2e-3.  Bound used here: 5e-3."""
    wl, d, run, _ = cfg0
    ctx = make_ctx(wl, precision=1)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    ref = run(wl.params, d)
    got = ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))
    check_mixed(got, ref, "cfg0 mixed", tol=5e-3)
    again = ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))
    assert all(torch_cuda.equal(a, b) for a, b in zip(got, again))
    ctx.destroy()


def test_cfg2_scaled_mixed_precision_parity(orc, torch_cuda):
    """config-2 recipe at 1/16 of the grid, noisy data, 600 walkers, FP32-accumulate variant."""
    wl = wlm.make_workload(2, n_w=600, t_obs=31557600.0 / 16)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl, precision=1)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    ref = run(wl.params, d)
    got = ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))
    check_mixed(got, ref, "cfg2/16 mixed")
    ctx.destroy()


def test_cfg2_full_size_sampled_mixed(orc, torch_cuda):
    """BASELINE.json config 2 at full size, FP32-accumulate variant, sampled walkers against the oracle."""
    wl = wlm.make_workload(2)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl, precision=1)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))]
    fis = np.array([orc.standin_fisco(p) for p in wl.params])
    sample = sorted({0, int(fis.argmin()), int(fis.argmax()), 1, 4097, 16383} | set(range(37, 16384, 2048)))
    ref = run(wl.params[sample], d)
    check_mixed([x[sample] for x in got], ref, "cfg2 mixed sampled")
    assert np.all(np.isfinite(got[0]))
    ctx.destroy()


def test_mixed_precision_multimode_is_unsupported(torch_cuda):
    from paper_2111_01064_b200 import binding
    wl = wlm.make_workload(3, n_w=8, t_obs=2.0 ** 16, n_knots=24)
    wl.f_nodes = wlm.geomspace_exact(wlm.F_LO, wlm.F_HI, 64)
    ctx = make_ctx(wl, precision=1)
    g = wl.grid
    z = torch_cuda.zeros(2 * g.n_f * 2, dtype=torch_cuda.float64, device="cuda")
    ctx.set_data(g.n_f, g.k_min, g.df, z, dev(torch_cuda, wl.W))
    with pytest.raises(binding.LLError) as ei:
        ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))
    assert ei.value.code == binding.LL_ERR_UNSUPPORTED
    ctx.destroy()


# ------------------------------------------------------------------------------------------- heterodyne
@pytest.fixture(scope="module")
def het_small(orc, torch_cuda):
    wl = wlm.make_workload(1, n_w=300, t_obs=2.0 ** 18, n_knots=37)
    d, h0, h0e, summ = oracle_setup_het(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    ctx.het_prepare(wl.f_edges, dev(torch_cuda, h0), dev(torch_cuda, h0e))
    return wl, d, h0, h0e, summ, ctx


def test_het_summary_data_matches_oracle(het_small):
    wl, d, h0, h0e, summ, ctx = het_small
    got = ctx.het_get_summary()
    for k in ("A0", "B0"):
        np.testing.assert_allclose(got[k], summ[k], rtol=1e-11, atol=1e-11 * np.abs(summ[k]).max(), err_msg=k)
    for k in ("A1", "B1"):      # first moments about the bin centre: cancel, so the scale is |.|_max
        np.testing.assert_allclose(got[k], summ[k], rtol=0, atol=1e-10 * np.abs(summ[k]).max(), err_msg=k)
    _, ddb = ctx.get_dd()
    assert abs(ddb - summ["dd_band"]) <= 1e-12 * summ["dd_band"]


def test_het_standin_parity(orc, het_small, torch_cuda):
    wl, d, h0, h0e, summ, ctx = het_small
    ref = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, wl.f_edges, h0e, summ)
    got = ctx.het_batch_standin(dev(torch_cuda, wl.params))
    check_triplet(got, ref, "het standin")


def test_het_arrays_parity(orc, het_small, torch_cuda):
    wl, d, h0, h0e, summ, ctx = het_small
    amp, ph, tf, _ = orc.standin_nodes(wl.params, wl.modes_m, wl.c_lm, wl.kappa, wl.f_edges,
                                       float(wl.f_edges[0]), float(wl.f_edges[-1]))
    ref = orc.het_batch(wl.f_edges, amp, ph, tf, h0e, summ)
    got = ctx.het_batch(dev(torch_cuda, amp), dev(torch_cuda, ph), dev(torch_cuda, tf))
    check_triplet(got, ref, "het arrays")


def test_het_equals_full_at_reference(het_small, torch_cuda):
    """north_star invariant: h = h0 => r = 1 => het log L = -1/2 <d-h0|d-h0> over the band."""
    wl, d, h0, h0e, summ, ctx = het_small
    logL, d_h, h_h = ctx.het_batch_standin(dev(torch_cuda, wl.inj[None]))
    f = wl.grid.freqs()
    m = (f >= wl.f_edges[0]) & (f <= wl.f_edges[-1])
    res = d[:, m, :] - h0[:, m, :]
    direct = -0.5 * float((wl.W[m][None, :] * (res ** 2).sum(axis=2)).sum())
    assert abs(float(logL[0]) - direct) <= 1e-6 * max(1.0, abs(direct))


@pytest.mark.parametrize("n_w", [1, 33, 1000])
def test_het_ragged_batches(orc, het_small, torch_cuda, n_w):
    wl, d, h0, h0e, summ, ctx = het_small
    rng = np.random.default_rng(n_w)
    params = wl.params[rng.integers(0, wl.n_w, n_w)].copy()
    params[:, 2] += rng.normal(0, 5.0, n_w)
    ref = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, params, wl.f_edges, h0e, summ)
    got = ctx.het_batch_standin(dev(torch_cuda, params))
    check_triplet(got, ref, f"het ragged {n_w}")
    assert ctx.het_batch_standin(dev(torch_cuda, params[:0]))[0].numel() == 0


def test_het_rerun_is_bit_identical(het_small, torch_cuda):
    wl, d, h0, h0e, summ, ctx = het_small
    p = dev(torch_cuda, wl.params)
    a = [x.clone() for x in ctx.het_batch_standin(p)]
    b = ctx.het_batch_standin(p)
    for x, y in zip(a, b):
        assert torch_cuda.equal(x, y)


def test_het_reference_zero_is_an_error(het_small, torch_cuda):
    from paper_2111_01064_b200 import binding
    wl, d, h0, h0e, summ, ctx = het_small
    bad = h0e.copy()
    bad[1, 3, :] = 0.0
    ctx2 = make_ctx(wl)
    g = wl.grid
    ctx2.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    with pytest.raises(binding.LLError) as ei:
        ctx2.het_prepare(wl.f_edges, dev(torch_cuda, h0), dev(torch_cuda, bad))
    assert ei.value.code == binding.LL_ERR_REF_ZERO
    with pytest.raises(binding.LLError) as ei:
        ctx2.het_batch_standin(dev(torch_cuda, wl.params))
    assert ei.value.code == binding.LL_ERR_STATE
    ctx2.destroy()


def test_cfg1_full_size(orc, torch_cuda):
    """BASELINE.json config 1 in full: 4096 walkers, 128 bins, 2^22 s grid (209 296 bins), noisy."""
    wl = wlm.make_workload(1)
    d, h0, h0e, summ = oracle_setup_het(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    ctx.het_prepare(wl.f_edges, dev(torch_cuda, h0), dev(torch_cuda, h0e))
    got_s = ctx.het_get_summary()
    np.testing.assert_allclose(got_s["A0"], summ["A0"], rtol=0, atol=1e-11 * np.abs(summ["A0"]).max())
    np.testing.assert_allclose(got_s["B0"], summ["B0"], rtol=1e-11)
    ref = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, wl.f_edges, h0e, summ)
    got = ctx.het_batch_standin(dev(torch_cuda, wl.params))
    check_triplet(got, ref, "cfg1")
    ctx.destroy()


def test_cfg3_higher_modes_full_size_sampled(orc, torch_cuda):
    """BASELINE.json config 3: six modes, 256 bins, 32768 walkers on the GPU; the oracle recomputes every 16th."""
    wl = wlm.make_workload(3)
    d, h0, h0e, summ = oracle_setup_het(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    ctx.het_prepare(wl.f_edges, dev(torch_cuda, h0), dev(torch_cuda, h0e))
    got = [x.cpu().numpy() for x in ctx.het_batch_standin(dev(torch_cuda, wl.params))]
    sample = np.arange(0, wl.n_w, 16)
    ref = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params[sample], wl.f_edges, h0e, summ)
    check_triplet([torch_cuda.as_tensor(x[sample]) for x in got], ref, "cfg3 sampled")
    assert np.all(np.isfinite(got[0]))
    ctx.destroy()


def test_cfg4_large_batch_full_size_sampled(orc, torch_cuda):
    """BASELINE.json config 4: 131072 walkers (16 x 8192), 512 bins; the oracle recomputes every 32nd walker."""
    wl = wlm.make_workload(4)
    d, h0, h0e, summ = oracle_setup_het(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    ctx.het_prepare(wl.f_edges, dev(torch_cuda, h0), dev(torch_cuda, h0e))
    got = [x.cpu().numpy() for x in ctx.het_batch_standin(dev(torch_cuda, wl.params))]
    sample = np.arange(0, wl.n_w, 32)
    ref = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params[sample], wl.f_edges, h0e, summ)
    check_triplet([torch_cuda.as_tensor(x[sample]) for x in got], ref, "cfg4 sampled")
    assert np.all(np.isfinite(got[0]))
    ctx.destroy()


# ------------------------------------------------------------------------------------------- boundary behaviour
def test_state_and_argument_errors(torch_cuda):
    from paper_2111_01064_b200 import binding
    ctx = binding.Context(n_modes=1)
    f_nodes = wlm.geomspace_exact(1e-4, 0.05, 16)
    p = torch_cuda.zeros((4, 9), dtype=torch_cuda.float64, device="cuda")
    with pytest.raises(binding.LLError) as ei:
        ctx.full_batch_standin(f_nodes, p)
    assert ei.value.code == binding.LL_ERR_STATE            # no data yet
    grid = wlm.make_grid(2.0 ** 14)
    W = dev(torch_cuda, wlm.trapezoid_weights(grid))
    d = torch_cuda.zeros((2, grid.n_f, 2), dtype=torch_cuda.float64, device="cuda")
    ctx.set_data(grid.n_f, grid.k_min, grid.df, d, W)
    with pytest.raises(binding.LLError) as ei:
        ctx.full_batch_standin(f_nodes, p)
    assert ei.value.code == binding.LL_ERR_STATE            # no stand-in description yet
    ctx.standin_config([2], [2], [1.0], 0.5)
    for bad in (f_nodes[::-1].copy(), f_nodes[:2], np.linspace(1e-3, 2e-3, 16)):
        with pytest.raises(binding.LLError) as ei:
            ctx.full_batch_standin(bad, p)
        assert ei.value.code == binding.LL_ERR_ARG
    with pytest.raises(binding.LLError) as ei:
        ctx.het_batch_standin(p)
    assert ei.value.code == binding.LL_ERR_STATE
    with pytest.raises(binding.LLError) as ei:
        ctx.set_data(0, grid.k_min, grid.df, d, W)
    assert ei.value.code == binding.LL_ERR_ARG
    # the entry points added for the SURVEY 8(f) rows: state before ll_het_prepare, sizes, NULLs
    tc = torch_cuda
    z = lambda *sh: tc.zeros(sh, dtype=tc.float64, device="cuda")
    for call in (lambda: ctx.het_audit_standin(p),
                 lambda: ctx.pt_stretch_half(0, z(1, 4, 9), z(1, 4), None, None, z(1), z(9), z(9), 5, z(1, 2), z(1, 2), z(1, 2))):
        with pytest.raises(binding.LLError) as ei:
            call()
        assert ei.value.code == binding.LL_ERR_STATE        # no heterodyne reference yet
    for call in (lambda: ctx.pt_stretch_half(2, z(1, 4, 9), z(1, 4), None, None, z(1), z(9), z(9), 5, z(1, 2), z(1, 2), z(1, 2)),
                 lambda: ctx.pt_stretch_half(0, z(1, 5, 9), z(1, 5), None, None, z(1), z(9), z(9), 5, z(1, 2), z(1, 2), z(1, 2)),
                 lambda: ctx.pt_stretch_half(0, z(1, 4, 9), z(1, 4), None, None, z(1), z(9), z(9), 0, z(1, 2), z(1, 2), z(1, 2)),
                 lambda: ctx.het_refresh_standin(p, z(4), 1),
                 lambda: ctx.full_batch_pw(z(4, 2), z(4, 1, 2), z(4, 1, 2), z(4, 1, 2, 2)),
                 lambda: ctx.pt_stats(z(0), None, None)):
        with pytest.raises(binding.LLError) as ei:
            call()
        assert ei.value.code == binding.LL_ERR_ARG
    assert ctx.full_batch_pw(z(0, 8), z(0, 1, 8), z(0, 1, 8), z(0, 1, 2, 2))[0].numel() == 0     # empty batch: no-op
    ctx.pt_swap(z(1, 4, 9), z(1, 4), None, None, z(1), None)                                    # one temperature: no-op
    ctx.destroy()


def test_smoke_entry(torch_cuda):
    import __graft_entry__
    __graft_entry__.smoke()


# ------------------------------------------------------------- reference update and audit
def test_het_audit_parity(orc, het_small, torch_cuda):
    """brute-force dense log L over the heterodyne band against the oracle's"""
    from oracle import reference_update as ru
    wl, d, h0, h0e, summ, ctx = het_small
    g = wl.grid
    ref = ru.audit(wl.params[:64], wl.modes_m, wl.c_lm, wl.kappa, g.k_min, g.df, g.n_f, d, wl.W, wl.f_edges)
    got = ctx.het_audit_standin(dev(torch_cuda, wl.params[:64]))
    check_triplet(got, ref, "het audit")
    assert ctx.het_audit_standin(dev(torch_cuda, wl.params[:0]))[0].numel() == 0


def test_het_refresh_parity(orc, torch_cuda):
    """reference update on the device: same best walker, same edges, same summary data and the same log L for the
    whole population afterwards as the oracle's step-by-step update; het = audit at the new reference."""
    from oracle import reference_update as ru
    wl = wlm.make_workload(1, n_w=300, t_obs=2.0 ** 18, n_knots=37)
    d, h0, h0e, summ = oracle_setup_het(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    ctx.het_prepare(wl.f_edges, dev(torch_cuda, h0), dev(torch_cuda, h0e))
    p = dev(torch_cuda, wl.params)
    logL0 = ctx.het_batch_standin(p)[0]
    ref0 = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, wl.f_edges, h0e, summ)
    up = ru.reference_update(wl.params, ref0["logL"], wl.modes_m, wl.c_lm, wl.kappa, g.k_min, g.df, g.n_f, d, wl.W, 41)
    best, f_edges = ctx.het_refresh_standin(p, logL0, 41)
    assert best == up["best"]
    # numpy.geomspace itself carries a few ulp of log10/pow rounding; the library forms the edges in long double
    np.testing.assert_allclose(f_edges, up["f_edges"], rtol=4e-15)
    assert f_edges[0] == up["f_edges"][0] and abs(f_edges[-1] / up["f_edges"][-1] - 1.0) <= 1e-15   # f_ISCO: pow(eta, -0.6) and the division, a few ulp
    # summary data: the library's own edges differ from numpy's by <= 2 ulp, which can move a dense bin across an
    # edge only if it sits on one; compare with the oracle run on the library's edges (edges are an input of H0)
    f = g.freqs()
    h0n = orc.standin_direct(wl.params[best], wl.modes_m, wl.c_lm, wl.kappa, f, float(f[0]), float(f[-1]))
    h0en = orc.standin_direct(wl.params[best], wl.modes_m, wl.c_lm, wl.kappa, f_edges, float(f[0]), float(f[-1]))
    summ_n = orc.het_prepare(g.k_min, g.df, d, wl.W, h0n, f_edges)
    got_s = ctx.het_get_summary()
    for k in ("A0", "B0"):
        np.testing.assert_allclose(got_s[k], summ_n[k], rtol=1e-10, atol=1e-10 * np.abs(summ_n[k]).max(), err_msg=k)
    ref = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, f_edges, h0en, summ_n)
    got = ctx.het_batch_standin(p)
    check_triplet(got, ref, "het after refresh")
    aud = ctx.het_audit_standin(p[best:best + 1])
    assert abs(float(got[0][best]) - float(aud[0][0])) <= 1e-6 * max(1.0, abs(float(aud[0][0])))
    # no finite log L -> error, state untouched
    from paper_2111_01064_b200 import binding
    with pytest.raises(binding.LLError):
        ctx.het_refresh_standin(p, torch_cuda.full_like(logL0, float("nan")), 41)
    ctx.destroy()


# ------------------------------------------------------------------- sampler step (R25-R28)
def _oracle_loglike_het(orc, wl, h0e, summ):
    def f(rows):
        r = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, rows, wl.f_edges, h0e, summ)
        return r["logL"], {"d_h": r["d_h"], "h_h": r["h_h"]}
    return f


def _prior_box(wl, params, widen):
    """uniform box around the population (Table I priors are uniform); the transfer factors are frozen"""
    P = params.shape[1]
    lo, hi = np.full(P, -np.inf), np.full(P, np.inf)
    c, w = params[:, :5].mean(axis=0), widen * np.ptp(params[:, :5], axis=0)
    lo[:5], hi[:5] = c - w, c + w
    return lo, hi


def test_pt_step_parity_het(orc, het_small, torch_cuda):
    """three iterations (two half updates + a swap sweep each) of 3 temperatures x 64 walkers on the heterodyned
    likelihood: same accept/swap decisions, same positions bit for bit, same log L within the FP64 bar."""
    from oracle import sampler as sm
    wl, d, h0, h0e, summ, ctx = het_small
    tc = torch_cuda
    rng = np.random.default_rng(190)
    n_t, n_w = 3, 64
    x = wl.params[:n_t * n_w].reshape(n_t, n_w, -1).copy()
    x[:, :, 5:] = wl.inj[5:]                                   # frozen coordinates: identical in every walker
    betas = np.array([1.0, 0.3, 0.05])
    lo, hi = _prior_box(wl, wl.params, 0.35)                   # tight enough that some proposals leave the box
    ll = _oracle_loglike_het(orc, wl, h0e, summ)
    l0, ex = ll(x.reshape(n_t * n_w, -1))
    logL, d_h, h_h = (v.reshape(n_t, n_w).copy() for v in (l0, ex["d_h"], ex["h_h"]))
    gx, gl, gd, gh = dev(tc, x), dev(tc, logL), dev(tc, d_h), dev(tc, h_h)
    gb, glo, ghi = dev(tc, betas), dev(tc, lo), dev(tc, hi)
    acc_g = tc.empty((n_t, n_w // 2), dtype=tc.int32, device="cuda")
    sw_g = tc.empty((n_t - 1, n_w), dtype=tc.int32, device="cuda")
    n_acc = n_out = n_sw = 0
    for it in range(3):
        for half in (0, 1):
            u = rng.random((3, n_t, n_w // 2))
            acc, y, ly, extra = sm.stretch_half(x, logL, half, betas, lo, hi, 5, 2.0, u[0], u[1], u[2], ll)
            k0 = 0 if half == 0 else n_w // 2                  # the oracle keeps d_h, h_h of accepted proposals too
            for t in range(n_t):
                sel = np.nonzero(acc[t])[0]
                d_h[t, k0 + sel] = extra["d_h"].reshape(n_t, -1)[t, sel]
                h_h[t, k0 + sel] = extra["h_h"].reshape(n_t, -1)[t, sel]
            ctx.pt_stretch_half(half, gx, gl, gd, gh, gb, glo, ghi, 5, dev(tc, u[0]), dev(tc, u[1]), dev(tc, u[2]),
                                accepted=acc_g)
            assert np.array_equal(acc_g.cpu().numpy().astype(bool), acc), f"accept decisions, it {it} half {half}"
            n_acc += int(acc.sum())
            n_out += int((~np.all((y >= lo) & (y <= hi), axis=2)).sum())
        us = rng.random((n_t - 1, n_w))
        done = sm.temperature_swaps(x, logL, betas, us)
        for t in range(n_t - 1, 0, -1):                          # d_h, h_h travel with the walker
            for i in np.nonzero(done[t - 1])[0]:
                d_h[t, i], d_h[t - 1, i] = d_h[t - 1, i], d_h[t, i]
                h_h[t, i], h_h[t - 1, i] = h_h[t - 1, i], h_h[t, i]
        ctx.pt_swap(gx, gl, gd, gh, gb, dev(tc, us), swapped=sw_g)
        assert np.array_equal(sw_g.cpu().numpy().astype(bool), done)
        n_sw += int(done.sum())
        assert np.array_equal(gx.cpu().numpy(), x), "positions are the same IEEE expression on both sides"
        check_triplet((gl.reshape(-1), gd.reshape(-1), gh.reshape(-1)),
                      {"logL": logL.reshape(-1), "d_h": d_h.reshape(-1), "h_h": h_h.reshape(-1)}, f"pt state it {it}")
    assert n_acc > 50 and n_out > 5 and n_sw > 5                # every branch was exercised
    best, bi, snr = sm.population_stats(logL, d_h, h_h)
    got = ctx.pt_stats(gl, gd, gh).cpu().numpy()
    assert int(got[1]) == bi and abs(got[0] - best) <= 1e-6 * max(1.0, abs(best)) and abs(got[2] - snr) <= 1e-9 * snr


def test_pt_step_parity_full(orc, torch_cuda):
    """the same move on the full-grid likelihood (Module 1): one iteration, 2 temperatures x 32 walkers"""
    from oracle import sampler as sm
    tc = torch_cuda
    wl = wlm.make_workload(0)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    rng = np.random.default_rng(194)
    n_t, n_w = 2, 32
    x = wl.params[:n_t * n_w].reshape(n_t, n_w, -1).copy()
    x[:, :, 5:] = wl.params[0, 5:]

    def ll(rows):
        r = run(rows, d)
        return r["logL"], {"d_h": r["d_h"], "h_h": r["h_h"]}
    betas = np.array([1.0, 0.01])
    lo, hi = _prior_box(wl, wl.params, 0.6)
    l0, _ = ll(x.reshape(n_t * n_w, -1))
    logL = l0.reshape(n_t, n_w).copy()
    gx, gl = dev(tc, x), dev(tc, logL)
    acc_g = tc.empty((n_t, n_w // 2), dtype=tc.int32, device="cuda")
    for half in (0, 1):
        u = rng.random((3, n_t, n_w // 2))
        acc, _, _, _ = sm.stretch_half(x, logL, half, betas, lo, hi, 5, 2.0, u[0], u[1], u[2], ll)
        ctx.pt_stretch_half(half, gx, gl, None, None, dev(tc, betas), dev(tc, lo), dev(tc, hi), 5, dev(tc, u[0]),
                            dev(tc, u[1]), dev(tc, u[2]), accepted=acc_g, f_nodes=wl.f_nodes)
        assert np.array_equal(acc_g.cpu().numpy().astype(bool), acc)
    assert np.array_equal(gx.cpu().numpy(), x)
    err = np.abs(gl.cpu().numpy() - logL) / np.maximum(1.0, np.abs(logL))
    assert err.max() <= 1e-6
    ctx.destroy()


def test_stop_functions_match_oracle():
    from oracle import sampler as sm
    from paper_2111_01064_b200 import binding
    assert binding.stop_snr(20.0, 20.0) and not binding.stop_snr(19.99, 20.0)
    st, ref = binding.StopState(n_checks=3, tol=1.0), sm.StopConverged(3, 1.0)
    for v in [-10.0, -5.0, -4.5, -4.2, -3.9, -2.0, -1.9, -1.8, -1.7, -1.65]:
        assert binding.stop_converged(st, v) == ref.check(v)


# ------------------------------------------------------------ per-walker node grids
@pytest.mark.parametrize("n_m,banded,n_w,n_nodes", [(1, False, 40, 33), (1, True, 97, 64), (3, True, 50, 20), (1, False, 1500, 48)])
def test_full_per_walker_nodes(orc, torch_cuda, n_m, banded, n_w, n_nodes):
    from oracle import per_walker as pw
    from paper_2111_01064_b200 import binding
    from helpers import pw_case
    tc = torch_cuda
    rng = np.random.default_rng(1000 * n_m + n_w)
    n_f, k_min, df = 5000, 40, 1e-5
    f, x, amp, ph, tf, W, d = pw_case(rng, n_w, n_m, n_nodes, n_f, k_min, df)
    band = np.stack([x[:, 0] * rng.uniform(0.9, 1.2, n_w), x[:, -1] * rng.uniform(0.6, 1.2, n_w)], axis=1) if banded else None
    if banded:
        band[3] = [f[-1] * 2, f[-1] * 3]                          # a walker whose band misses the grid
    ctx = binding.Context(n_modes=n_m)
    ctx.set_data(n_f, k_min, df, dev(tc, d), dev(tc, W))
    got = ctx.full_batch_pw(dev(tc, x), dev(tc, amp), dev(tc, ph), dev(tc, tf), None if band is None else dev(tc, band))
    sample = np.arange(n_w) if n_w <= 100 else np.r_[0, 1, 31, 32, 1023, 1024, n_w - 1, rng.integers(0, n_w, 20)]
    ref = pw.full_batch_pw(x[sample], amp[sample], ph[sample], tf[sample], None if band is None else band[sample],
                           k_min, df, d, W)
    check_triplet([__import__("torch").as_tensor(v.cpu().numpy()[sample]) for v in got], ref, "per-walker nodes")
    if banded:
        dd_full, _ = ctx.get_dd()
        assert float(got[0][3]) == -0.5 * dd_full and float(got[2][3]) == 0.0
    # identical nodes for every walker: the per-walker path equals the shared-node path (needs nodes covering the grid)
    xs = np.tile(np.geomspace(f[0] * 0.9, f[-1] * 1.05, n_nodes), (n_w, 1))
    a = ctx.full_batch_pw(dev(tc, xs), dev(tc, amp), dev(tc, ph), dev(tc, tf))
    b = ctx.full_batch(xs[0], dev(tc, amp), dev(tc, ph), dev(tc, tf))
    for u, v in zip(a, b):
        un, vn = u.cpu().numpy(), v.cpu().numpy()
        assert np.all(np.abs(un - vn) <= 1e-9 * np.maximum(1.0, np.abs(vn)))
    ctx.destroy()


def test_set_data_again_invalidates_cached_tiles(orc, torch_cuda):
    """ll_set_data "may be called again at any time" (include/ll.h): a second data stream with MORE bins in the same
    tile-size bucket must not reuse the frequency-tile table of the first (the per-walker path never rebuilds the node
    tables, so nothing else would invalidate it), and alternating per-walker and shared-node calls must stay right."""
    from oracle import per_walker as pw
    from paper_2111_01064_b200 import binding
    from helpers import pw_case
    tc = torch_cuda
    rng = np.random.default_rng(312)
    k_min, df, n_w, n_nodes = 40, 1e-5, 40, 33
    ctx = binding.Context(n_modes=1)
    for n_f in (3000, 5000, 4000):
        f, x, amp, ph, tf, W, d = pw_case(rng, n_w, 1, n_nodes, n_f, k_min, df)
        ctx.set_data(n_f, k_min, df, dev(tc, d), dev(tc, W))
        got = ctx.full_batch_pw(dev(tc, x), dev(tc, amp), dev(tc, ph), dev(tc, tf))
        ref = pw.full_batch_pw(x, amp, ph, tf, None, k_min, df, d, W)
        check_triplet(got, ref, f"per-walker nodes after set_data(n_f={n_f})")
        xs = np.geomspace(f[0] * 0.9, f[-1] * 1.05, n_nodes)
        got = ctx.full_batch(xs, dev(tc, amp), dev(tc, ph), dev(tc, tf))
        ref = orc.full_batch(xs, amp, ph, tf, None, k_min, df, d, W)
        check_triplet(got, ref, f"shared nodes after set_data(n_f={n_f})")
        got = ctx.full_batch_pw(dev(tc, x), dev(tc, amp), dev(tc, ph), dev(tc, tf))
        check_triplet(got, pw.full_batch_pw(x, amp, ph, tf, None, k_min, df, d, W), "per-walker nodes, alternating")
    ctx.destroy()


# ------------------------------------------------------- not-a-knot boundary condition
@pytest.fixture
def notaknot(orc):
    orc.set_spline_bc(1)
    yield orc
    orc.set_spline_bc(0)


def test_notaknot_all_spline_kernels(notaknot, torch_cuda):
    """ll_config.spline_bc = LL_BC_NOT_A_KNOT through every spline kernel: block-per-system (small batch), thread-per-
    system (large batch), six-spline transfer-function path, per-walker nodes; oracle under the same switch."""
    from oracle import per_walker as pw
    from paper_2111_01064_b200 import binding
    from helpers import pw_case
    orc, tc = notaknot, torch_cuda
    # stand-in entry point, config-0 recipe (small batch -> k_spline_block)
    wl = wlm.make_workload(0)
    d, run = oracle_setup_full(orc, wl)                    # data = walker 0's NOT-A-KNOT spline template
    ctx = binding.Context(n_modes=1, spline_bc=binding.LL_BC_NOT_A_KNOT)
    ctx.standin_config(wl.modes_l, wl.modes_m, wl.c_lm, wl.kappa)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    got = ctx.full_batch_standin(wl.f_nodes, dev(tc, wl.params))
    check_triplet(got, run(wl.params, d), "not-a-knot cfg0")
    assert abs(float(got[0][0])) <= 1e-6                   # log L = 0 at d = h under this BC too
    with pytest.raises(binding.LLError):
        ctx.tlm_nodes(wl.f_nodes, dev(tc, np.zeros((1, 1, len(wl.f_nodes)))), 0.0)
    ctx.destroy()
    # array entry points on a random grid: large batch (thread-per-system), transfer-function path, per-walker nodes
    rng = np.random.default_rng(2)
    n_f, k_min, df = 3000, 40, 1e-5
    f, x, amp, ph, tf, W, dd_ = pw_case(rng, 5000, 1, 24, n_f, k_min, df)
    xs = np.geomspace(f[0] * 0.95, f[-1] * 1.02, 24)
    ctx = binding.Context(n_modes=1, spline_bc=binding.LL_BC_NOT_A_KNOT)
    ctx.set_data(n_f, k_min, df, dev(tc, dd_), dev(tc, W))
    got = ctx.full_batch(xs, dev(tc, amp), dev(tc, ph), dev(tc, tf))
    sample = np.r_[0, 1, 4999, rng.integers(0, 5000, 30)]
    ref = orc.full_batch(xs, amp[sample], ph[sample], tf[sample], None, k_min, df, dd_, W)
    check_triplet([__import__("torch").as_tensor(v.cpu().numpy()[sample]) for v in got], ref, "not-a-knot large batch")
    s2 = sample[:12]
    tfn = _smooth_tf_nodes(rng, len(s2), 1, xs)
    got = ctx.full_batch_tf(xs, dev(tc, amp[s2]), dev(tc, ph[s2]), dev(tc, tfn))
    check_triplet(got, orc.full_batch_tf(xs, amp[s2], ph[s2], tfn, None, k_min, df, dd_, W), "not-a-knot tf")
    got = ctx.full_batch_pw(dev(tc, x[:200]), dev(tc, amp[:200]), dev(tc, ph[:200]), dev(tc, tf[:200]))
    check_triplet(got, pw.full_batch_pw(x[:200], amp[:200], ph[:200], tf[:200], None, k_min, df, dd_, W), "not-a-knot per-walker")
    # and the boundary condition really changes the answer
    ctx_n = binding.Context(n_modes=1)
    ctx_n.set_data(n_f, k_min, df, dev(tc, dd_), dev(tc, W))
    nat = ctx_n.full_batch_pw(dev(tc, x[:200]), dev(tc, amp[:200]), dev(tc, ph[:200]), dev(tc, tf[:200]))
    assert float((nat[1] - got[1]).abs().max()) > 1e-6 * float(got[2].abs().max())
    ctx.destroy(); ctx_n.destroy()


def test_one_year_noiseless_logL_is_zero_at_truth(orc, torch_cuda):
    """The thinnest margin of the FP64 bar (SURVEY 8(c) probes): noiseless data on the one-year grid, log L = 0 at
    the injection to 1e-6 ABSOLUTE while <d|h> = <h|h> = <d|d> = 2.5e5 — each of them is needed to
    4e-12 relative.  Also a near walker and a far one against the oracle."""
    wl = wlm.make_workload(2)
    wl.noise = None
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    p = wl.params[:3].copy()
    p[1] = wl.inj
    p[1, 0] *= 1.0 + 3e-4                                   # near: log L of a few hundred
    p[1, 2] += 3.0
    ref = run(p, d)
    got = ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, p))
    check_triplet(got, ref, "one-year noiseless")
    assert abs(ref["logL"][0]) <= 1e-6 and abs(float(got[0][0])) <= 1e-6
    assert -1e4 < ref["logL"][1] < -10.0
    # the same through a large batch (other tiles, thread-per-system spline)
    big = np.tile(p, (2000, 1))
    gb = ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, big))[0].cpu().numpy().reshape(2000, 3)
    assert np.all(np.abs(gb - ref["logL"][None, :]) <= 1e-6 * np.maximum(1.0, np.abs(ref["logL"]))[None, :])
    ctx.destroy()


def test_pt_run_parity_het(orc, het_small, torch_cuda):
    """ll_pt_run_het: 12 whole iterations with the counter-based uniforms (reading R31) against the oracle's loop with
    its own implementation of the same generator: identical positions, acceptance counts, log L at the FP64 bar;
    two runs of 6 continue exactly like one run of 12."""
    from oracle import sampler as sm
    wl, d, h0, h0e, summ, ctx = het_small
    tc = torch_cuda
    n_t, n_w = 3, 64
    x = wl.params[:n_t * n_w].reshape(n_t, n_w, -1).copy()
    x[:, :, 5:] = wl.inj[5:]
    betas = np.array([1.0, 0.3, 0.05])
    lo, hi = _prior_box(wl, wl.params, 0.35)
    ll = _oracle_loglike_het(orc, wl, h0e, summ)
    logL = ll(x.reshape(n_t * n_w, -1))[0].reshape(n_t, n_w).copy()
    gx, gl = dev(tc, x), dev(tc, logL)
    gx2, gl2 = gx.clone(), gl.clone()
    acc_g = tc.zeros(n_t, dtype=tc.int64, device="cuda")
    seed = 2111_01064
    n_acc = sm.run(x, logL, betas, lo, hi, 5, 2.0, seed, 100, 12, ll)
    ctx.pt_run(gx, gl, None, None, dev(tc, betas), dev(tc, lo), dev(tc, hi), 5, seed, 100, 12, n_accepted=acc_g)
    assert np.array_equal(gx.cpu().numpy(), x)
    assert np.array_equal(acc_g.cpu().numpy(), n_acc) and n_acc.sum() > 200
    err = np.abs(gl.cpu().numpy() - logL) / np.maximum(1.0, np.abs(logL))
    assert err.max() <= 1e-6
    ctx.pt_run(gx2, gl2, None, None, dev(tc, betas), dev(tc, lo), dev(tc, hi), 5, seed, 100, 6)
    ctx.pt_run(gx2, gl2, None, None, dev(tc, betas), dev(tc, lo), dev(tc, hi), 5, seed, 106, 6)
    assert tc.equal(gx2, gx) and tc.equal(gl2, gl)


def test_pt_run_fused_150_iterations_and_both_forms(orc, het_small, torch_cuda):
    """ll_pt_run_het as ONE cooperative launch (k_pt_run_het1: the whole loop on the device, grid barriers between the
    half updates and the swap sweep): 150 iterations (the paper's check cadence) against the oracle's
    loop — identical positions, equal acceptance counters — and against the 9-launches-per-iteration form of the same
    entry point (ll_pt_fused(0)): same positions, log L equal to rounding."""
    from oracle import sampler as sm
    wl, d, h0, h0e, summ, ctx = het_small
    tc = torch_cuda
    n_t, n_w = 3, 64
    x = wl.params[:n_t * n_w].reshape(n_t, n_w, -1).copy()
    x[:, :, 5:] = wl.inj[5:]
    betas = np.array([1.0, 0.3, 0.05])
    lo, hi = _prior_box(wl, wl.params, 0.35)
    ll = _oracle_loglike_het(orc, wl, h0e, summ)
    logL = ll(x.reshape(n_t * n_w, -1))[0].reshape(n_t, n_w).copy()
    out0 = ctx.het_batch_standin(dev(tc, x.reshape(n_t * n_w, -1)))
    gx, gl, gd, gh = dev(tc, x), dev(tc, logL), out0[1].reshape(n_t, n_w).clone(), out0[2].reshape(n_t, n_w).clone()
    ux, ul, ud, uh = gx.clone(), gl.clone(), gd.clone(), gh.clone()
    acc_g = tc.zeros(n_t, dtype=tc.int64, device="cuda")
    acc_u = tc.zeros(n_t, dtype=tc.int64, device="cuda")
    seed, n_iter = 2111, 150
    n_acc = sm.run(x, logL, betas, lo, hi, 5, 2.0, seed, 40, n_iter, ll)
    launches0 = ctx.kernel_launches()
    ctx.pt_run(gx, gl, gd, gh, dev(tc, betas), dev(tc, lo), dev(tc, hi), 5, seed, 40, n_iter, n_accepted=acc_g)
    assert ctx.kernel_launches() - launches0 == 1                       # the whole run is one launch
    assert np.array_equal(gx.cpu().numpy(), x)
    assert np.array_equal(acc_g.cpu().numpy(), n_acc) and n_acc.sum() > 5000
    err = np.abs(gl.cpu().numpy() - logL) / np.maximum(1.0, np.abs(logL))
    assert err.max() <= 1e-6
    # the carried <d|h>, <h|h> belong to the positions
    chk = ctx.het_batch_standin(gx.reshape(n_t * n_w, -1))
    assert np.allclose(gd.cpu().numpy().ravel(), chk[1].cpu().numpy(), rtol=1e-9, atol=1e-9)
    assert np.allclose(gh.cpu().numpy().ravel(), chk[2].cpu().numpy(), rtol=1e-9)
    ctx.pt_fused(False)
    try:
        launches0 = ctx.kernel_launches()
        ctx.pt_run(ux, ul, ud, uh, dev(tc, betas), dev(tc, lo), dev(tc, hi), 5, seed, 40, n_iter, n_accepted=acc_u)
        assert ctx.kernel_launches() - launches0 == 8 * n_iter          # uniforms, 2 x (propose, H1-H3, accept), swaps
    finally:
        ctx.pt_fused(True)
    assert tc.equal(ux, gx) and tc.equal(acc_u, acc_g)
    assert np.allclose(ul.cpu().numpy(), gl.cpu().numpy(), rtol=1e-12, atol=1e-9)


def test_pt_run_fused_module2_size(orc, torch_cuda):
    """Module-2 size (10 temperatures x 400 walkers) on the config-1 recipe: the one-launch loop and the
    multi-launch loop end at the same positions after 40 iterations; sampled log L against the oracle."""
    tc = torch_cuda
    wl = wlm.make_workload(1, n_w=4000, t_obs=2.0 ** 18, n_knots=128)
    d, h0, h0e, summ = oracle_setup_het(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    ctx.het_prepare(wl.f_edges, dev(tc, h0), dev(tc, h0e))
    n_t, n_w = 10, 400
    x = wl.params.reshape(n_t, n_w, -1).copy()
    x[:, :, 5:] = wl.inj[5:]
    betas = np.array([0.5 ** t for t in range(n_t - 1)] + [0.0])
    lo, hi = _prior_box(wl, wl.params, 3.0)
    gx = dev(tc, x)
    out0 = ctx.het_batch_standin(gx.reshape(n_t * n_w, -1))
    gl, gd, gh = (v.reshape(n_t, n_w).clone() for v in out0)
    ux, ul, ud, uh = gx.clone(), gl.clone(), gd.clone(), gh.clone()
    args = (dev(tc, betas), dev(tc, lo), dev(tc, hi), 5, 77, 0, 40)
    acc_g = tc.zeros(n_t, dtype=tc.int64, device="cuda")
    acc_u = tc.zeros(n_t, dtype=tc.int64, device="cuda")
    ctx.pt_run(gx, gl, gd, gh, *args, n_accepted=acc_g)
    ctx.pt_fused(False)
    ctx.pt_run(ux, ul, ud, uh, *args, n_accepted=acc_u)
    ctx.pt_fused(True)
    assert tc.equal(ux, gx) and tc.equal(acc_u, acc_g) and int(acc_g.sum()) > 0.2 * 40 * n_t * n_w
    assert not tc.equal(gx, dev(tc, x))
    sample = np.r_[0:8, 1990:2010, 3990:4000]
    rows = gx.reshape(n_t * n_w, -1).cpu().numpy()[sample]
    ref = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, rows, wl.f_edges, h0e, summ)
    got = gl.reshape(-1).cpu().numpy()[sample]
    assert np.all(np.abs(got - ref["logL"]) <= 1e-6 * np.maximum(1.0, np.abs(ref["logL"])))
    ctx.destroy()


def test_module2_loop_with_reference_update(orc, torch_cuda):
    """The Module-2 loop in miniature: sample, update the reference to the best walker, re-evaluate
    the population against the new reference, sample on, read the stopping statistics — library calls only on one
    side, the oracle's step-by-step functions on the other; identical walker positions at the end."""
    from oracle import sampler as sm
    from paper_2111_01064_b200 import binding
    tc = torch_cuda
    wl = wlm.make_workload(1, n_w=128, t_obs=2.0 ** 18, n_knots=37)
    d, h0, h0e, summ = oracle_setup_het(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    f = g.freqs()
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    ctx.het_prepare(wl.f_edges, dev(tc, h0), dev(tc, h0e))
    n_t, n_w = 2, 64
    x = wl.params.reshape(n_t, n_w, -1).copy()
    x[:, :, 5:] = wl.inj[5:]
    betas = np.array([1.0, 0.2])
    lo, hi = _prior_box(wl, wl.params, 0.5)
    seed = 5000
    # ---- oracle side
    edges, he, sm_ = wl.f_edges, h0e, summ
    ll = lambda rows: (orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, rows, edges, he, sm_)["logL"], {})
    xo = x.copy()
    lo_ = ll(xo.reshape(n_t * n_w, -1))[0].reshape(n_t, n_w).copy()
    sm.run(xo, lo_, betas, lo, hi, 5, 2.0, seed, 0, 10, ll)
    # ---- library side, first block
    gx = dev(tc, x)
    out = ctx.het_batch_standin(gx.reshape(n_t * n_w, -1))
    gl, gd, gh = (v.reshape(n_t, n_w).clone() for v in out)
    gb, glo, ghi = dev(tc, betas), dev(tc, lo), dev(tc, hi)
    ctx.pt_run(gx, gl, gd, gh, gb, glo, ghi, 5, seed, 0, 10)
    assert np.array_equal(gx.cpu().numpy(), xo)
    # ---- reference update on both sides (the library's edges are an input of the oracle's H0, cf. test_het_refresh_parity)
    best, f_edges = ctx.het_refresh_standin(gx.reshape(n_t * n_w, -1), gl.reshape(-1), 38)
    assert best == sm.population_stats(lo_, lo_, np.ones_like(lo_))[1]
    pb = xo.reshape(n_t * n_w, -1)[best]
    h0n = orc.standin_direct(pb, wl.modes_m, wl.c_lm, wl.kappa, f, float(f[0]), float(f[-1]))
    he = orc.standin_direct(pb, wl.modes_m, wl.c_lm, wl.kappa, f_edges, float(f[0]), float(f[-1]))
    sm_ = orc.het_prepare(g.k_min, g.df, d, wl.W, h0n, f_edges)
    edges = f_edges
    lo_ = ll(xo.reshape(n_t * n_w, -1))[0].reshape(n_t, n_w).copy()
    out = ctx.het_batch_standin(gx.reshape(n_t * n_w, -1))
    gl, gd, gh = (v.reshape(n_t, n_w).clone() for v in out)
    # ---- second block and the stopping statistics
    sm.run(xo, lo_, betas, lo, hi, 5, 2.0, seed, 10, 10, ll)
    ctx.pt_run(gx, gl, gd, gh, gb, glo, ghi, 5, seed, 10, 10)
    assert np.array_equal(gx.cpu().numpy(), xo)
    st = ctx.pt_stats(gl[0], gd[0], gh[0]).cpu().numpy()
    best_o, bi_o, _ = sm.population_stats(lo_[0], lo_[0], np.ones(n_w))
    assert int(st[1]) == bi_o and abs(st[0] - best_o) <= 1e-6 * max(1.0, abs(best_o))
    stop = binding.StopState(n_checks=30, tol=1.0)
    assert not binding.stop_converged(stop, float(st[0]))
    ctx.destroy()


def test_pt_run_parity_full(orc, torch_cuda):
    """ll_pt_run_full: three whole iterations on the full-grid likelihood (Module 1) with the counter-based
    uniforms, against the oracle's loop: identical positions and acceptance counts."""
    from oracle import sampler as sm
    tc = torch_cuda
    wl = wlm.make_workload(0)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    n_t, n_w = 2, 32
    x = wl.params[:n_t * n_w].reshape(n_t, n_w, -1).copy()
    x[:, :, 5:] = wl.params[0, 5:]
    ll = lambda rows: (run(rows, d)["logL"], {})
    betas = np.array([1.0, 0.01])
    lo, hi = _prior_box(wl, wl.params, 0.6)
    logL = ll(x.reshape(n_t * n_w, -1))[0].reshape(n_t, n_w).copy()
    gx, gl = dev(tc, x), dev(tc, logL)
    acc_g = tc.zeros(n_t, dtype=tc.int64, device="cuda")
    n_acc = sm.run(x, logL, betas, lo, hi, 5, 2.0, 194, 7, 3, ll)
    ctx.pt_run(gx, gl, None, None, dev(tc, betas), dev(tc, lo), dev(tc, hi), 5, 194, 7, 3, n_accepted=acc_g, f_nodes=wl.f_nodes)
    assert np.array_equal(gx.cpu().numpy(), x) and np.array_equal(acc_g.cpu().numpy(), n_acc) and n_acc.sum() > 10
    err = np.abs(gl.cpu().numpy() - logL) / np.maximum(1.0, np.abs(logL))
    assert err.max() <= 1e-6
    ctx.destroy()
