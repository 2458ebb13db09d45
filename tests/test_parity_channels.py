"""GPU parity tests (-m gpu) for the two SURVEY §8(f) completions of round 2, every kernel family against the oracle:
  * three TDI channels A, E, T with per-channel weights W [n_c][n_f] (Eq. 3 sums over A, E, T, "T different":
    PAPER.md:41, 67-70; reading R5), plus the two other weight layouts (two channels with their own rows; three
    channels sharing one row);
  * the linear phase term kept outside the spline, Psi_m(f) = spline_m(f) + 2 pi f t_shift (
    reading R32), on the array entry points and as the stand-in's own t_c (ll_standin_split_tc).
Tolerance: BASELINE.json north_star, as in test_parity_gpu.py."""
import numpy as np
import pytest

from paper_2111_01064_b200 import workloads as wlm
from helpers import (check_triplet, dev, make_ctx, oracle_setup_full, oracle_setup_het, pw_case, rand_smooth_nodes, unit_tf)

pytestmark = pytest.mark.gpu


def _weights(rng, grid, n_c, per_channel):
    """physical-scale weights: the workload PSDs times a channel-dependent random factor, so every row differs"""
    W = 4.0 * grid.df / wlm.channel_psds(grid.freqs(), n_c)
    W *= rng.uniform(0.5, 2.0, (n_c, 1))
    return np.ascontiguousarray(W if per_channel else W[0])


def _noise(rng, grid, n_c):
    sigma = np.sqrt(wlm.channel_psds(grid.freqs(), n_c) / (4 * grid.df))
    return rng.standard_normal((n_c, grid.n_f, 2)) * sigma[:, :, None]


def _smooth_tf_nodes(rng, n_w, n_m, f_nodes, n_c):
    x = np.log(f_nodes / f_nodes[0]) / np.log(f_nodes[-1] / f_nodes[0])
    a = rng.uniform(-1.0, 1.0, (n_w, n_m, n_c, 6, 1))
    mod = 1.0 + 0.3 * a[..., 0, :] * x + 0.2 * a[..., 1, :] * np.sin(2 * x + a[..., 2, :])
    ang = 3.0 * a[..., 3, :] + 2.0 * a[..., 4, :] * x
    return np.ascontiguousarray(np.stack([mod * np.cos(ang), mod * np.sin(ang)], axis=-1))


# --------------------------------------------------------------------------- array entry points, all weight layouts
@pytest.mark.parametrize("n_c,per_channel,n_m,n_w", [(3, True, 1, 97), (3, True, 3, 50), (2, True, 1, 70), (2, True, 2, 40),
                                                     (3, False, 1, 45), (3, True, 1, 1500)])
def test_full_arrays_channels_and_weight_rows(orc, torch_cuda, n_c, per_channel, n_m, n_w):
    """ll_full_batch, ll_full_batch_tf and ll_full_batch_pw with n_c channels and one weight row per channel (or one
    shared row): k_full_fused<1|0, NC, WS>, k_full_fused_tf, k_full_fused_pw, k_finalize against the oracle."""
    from oracle import per_walker as pw
    from paper_2111_01064_b200 import binding
    tc = torch_cuda
    rng = np.random.default_rng(7000 + 100 * n_c + 10 * n_m + n_w)
    grid = wlm.make_grid(2.0 ** 16)
    f = grid.freqs()
    f_nodes = wlm.geomspace_exact(wlm.F_LO, wlm.F_HI, 61)
    W = _weights(rng, grid, n_c, per_channel)
    amp, ph = rand_smooth_nodes(rng, n_w, n_m, f_nodes)
    tf = unit_tf(rng, n_w, n_m, n_c)
    d = _noise(rng, grid, n_c)
    lo = rng.uniform(0.5e-4, 5e-3, n_w)
    band = np.stack([lo, lo * rng.uniform(1.0, 40.0, n_w)], axis=1)
    band[0] = [f[10], f[10]]
    band[1] = [f[0], f[-1]]
    ctx = binding.Context(n_modes=n_m, n_channels=n_c)
    ctx.set_data(grid.n_f, grid.k_min, grid.df, dev(tc, d), dev(tc, W))
    assert abs(ctx.get_dd()[0] - orc.dd(d, W)) <= 1e-12 * orc.dd(d, W)
    sample = np.arange(n_w) if n_w <= 100 else np.unique(np.r_[0, 1, 31, 32, 127, 128, 1023, 1024, n_w - 1, rng.integers(0, n_w, 30)])
    pick = lambda got: [__import__("torch").as_tensor(v.cpu().numpy()[sample]) for v in got]
    got = ctx.full_batch(f_nodes, dev(tc, amp), dev(tc, ph), dev(tc, tf), dev(tc, band))
    ref = orc.full_batch(f_nodes, amp[sample], ph[sample], tf[sample], band[sample], grid.k_min, grid.df, d, W)
    check_triplet(pick(got), ref, f"arrays n_c={n_c} per_channel={per_channel} n_m={n_m}")
    again = ctx.full_batch(f_nodes, dev(tc, amp), dev(tc, ph), dev(tc, tf), dev(tc, band))
    assert all(tc.equal(a, b) for a, b in zip(got, again))
    if n_w > 1000:
        ctx.destroy()
        return
    # frequency-dependent transfer function (Eq. 8-9): 2 + 2 n_c splines per mode
    tfn = _smooth_tf_nodes(rng, n_w, n_m, f_nodes, n_c)
    got = ctx.full_batch_tf(f_nodes, dev(tc, amp), dev(tc, ph), dev(tc, tfn), dev(tc, band))
    ref = orc.full_batch_tf(f_nodes, amp, ph, tfn, band, grid.k_min, grid.df, d, W)
    check_triplet(got, ref, f"tf n_c={n_c} n_m={n_m}")
    # per-walker node grids
    x = np.stack([np.geomspace(f[0] * rng.uniform(0.8, 1.5), f[-1] * rng.uniform(0.4, 1.1), 48) for _ in range(n_w)])
    ampw, phw = (np.stack([rand_smooth_nodes(rng, 1, n_m, x[w])[k][0] for w in range(n_w)]) for k in (0, 1))
    got = ctx.full_batch_pw(dev(tc, x), dev(tc, ampw), dev(tc, phw), dev(tc, tf), dev(tc, band))
    ref = pw.full_batch_pw(x, ampw, phw, tf, band, grid.k_min, grid.df, d, W)
    check_triplet(got, ref, f"per-walker nodes n_c={n_c} n_m={n_m}")
    ctx.destroy()


def test_cfg0_three_channels_standin(orc, torch_cuda):
    """config-0 recipe with three channels (A, E, T; the T channel with its own PSD): stand-in entry point, log L[0] = 0,
    the dense template utility, ragged batch."""
    tc = torch_cuda
    wl = wlm.make_workload(0, n_c=3)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    ref = run(wl.params, d)
    got = ctx.full_batch_standin(wl.f_nodes, dev(tc, wl.params))
    check_triplet(got, ref, "cfg0 three channels")
    assert abs(float(got[0][0])) <= 1e-6 and np.sqrt(float(got[2][0])) == pytest.approx(500.0, rel=1e-9)
    h = ctx.full_template_standin(wl.f_nodes, wl.params[5]).cpu().numpy()
    href = run(wl.params[5][None], None, True)["h"]
    assert h.shape == (3, g.n_f, 2) and np.abs(h - href).max() <= 1e-9 * np.abs(href).max()
    got = ctx.full_batch_standin(wl.f_nodes, dev(tc, wl.params[:33]))
    check_triplet(got, run(wl.params[:33], d), "cfg0 three channels, 33 walkers")
    ctx.destroy()


def test_cfg2_scaled_three_channels(orc, torch_cuda):
    """config-2 recipe at 1/16 of the grid with three channels: several walker blocks and tiles, the large-batch route."""
    tc = torch_cuda
    wl = wlm.make_workload(2, n_w=1200, t_obs=31557600.0 / 16, n_c=3)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(tc, wl.params))]
    sample = np.r_[0:40, 1023:1030, 1190:1200]
    ref = run(wl.params[sample], d)
    check_triplet([__import__("torch").as_tensor(x[sample]) for x in got], ref, "cfg2/16 three channels")
    ctx.destroy()


# --------------------------------------------------------------------------- heterodyne, three channels
@pytest.mark.parametrize("index,n_w", [(1, 300), (3, 100)])
def test_het_three_channels(orc, torch_cuda, index, n_w):
    """config-1 (one mode: the edge-regrouped kernel) and config-3 (six modes) recipes with three channels and
    per-channel PSDs: summary data, stand-in and array entry points, brute-force audit."""
    from oracle import reference_update as ru
    tc = torch_cuda
    wl = wlm.make_workload(index, n_w=n_w, t_obs=2.0 ** 17, n_knots=40, n_c=3)
    d, h0, h0e, summ = oracle_setup_het(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    f = g.freqs()
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    ctx.het_prepare(wl.f_edges, dev(tc, h0), dev(tc, h0e))
    s = ctx.het_get_summary()
    for k in ("A0", "A1", "B0", "B1"):
        assert s[k].shape == summ[k].shape
        np.testing.assert_allclose(s[k], summ[k], rtol=1e-10, atol=1e-11 * np.abs(summ[k]).max(), err_msg=k)
    assert ctx.get_dd()[1] == pytest.approx(summ["dd_band"], rel=1e-12)
    ref = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, wl.f_edges, h0e, summ)
    got = ctx.het_batch_standin(dev(tc, wl.params))
    check_triplet(got, ref, f"het stand-in three channels cfg{index}")
    amp, ph, tf, _ = orc.standin_nodes(wl.params, wl.modes_m, wl.c_lm, wl.kappa, wl.f_edges, f[0], f[-1])
    got = ctx.het_batch(dev(tc, amp), dev(tc, ph), dev(tc, tf))
    check_triplet(got, orc.het_batch(wl.f_edges, amp, ph, tf, h0e, summ), f"het arrays three channels cfg{index}")
    got = ctx.het_audit_standin(dev(tc, wl.params[:24]))
    check_triplet(got, ru.audit(wl.params[:24], wl.modes_m, wl.c_lm, wl.kappa, g.k_min, g.df, g.n_f, d, wl.W, wl.f_edges),
                  f"audit three channels cfg{index}")
    if index == 1:
        logL = ctx.het_batch_standin(dev(tc, wl.params))[0]
        best, f_edges = ctx.het_refresh_standin(dev(tc, wl.params), logL, 41)
        up = ru.reference_update(wl.params, logL.cpu().numpy(), wl.modes_m, wl.c_lm, wl.kappa, g.k_min, g.df, g.n_f, d, wl.W, 41)
        assert best == up["best"]
        np.testing.assert_allclose(f_edges, up["f_edges"], rtol=1e-14)
        h0n = orc.standin_direct(wl.params[best], wl.modes_m, wl.c_lm, wl.kappa, f, f[0], f[-1])
        h0en = orc.standin_direct(wl.params[best], wl.modes_m, wl.c_lm, wl.kappa, f_edges, f[0], f[-1])
        sn = orc.het_prepare(g.k_min, g.df, d, wl.W, h0n, f_edges)
        ref = orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, f_edges, h0en, sn)
        check_triplet(ctx.het_batch_standin(dev(tc, wl.params)), ref, "het after the reference update, three channels")
    ctx.destroy()


def test_sampler_run_three_channels(orc, torch_cuda):
    """ll_pt_run_het on a three-channel population (rows of 11 doubles): identical positions and acceptance counts
    to the oracle's loop over 8 iterations."""
    from oracle import sampler as sm
    tc = torch_cuda
    wl = wlm.make_workload(1, n_w=128, t_obs=2.0 ** 17, n_knots=24, n_c=3)
    d, h0, h0e, summ = oracle_setup_het(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    ctx.het_prepare(wl.f_edges, dev(tc, h0), dev(tc, h0e))
    n_t, n_w = 2, 64
    x = wl.params.reshape(n_t, n_w, -1).copy()
    x[:, :, 5:] = wl.inj[5:]
    betas = np.array([1.0, 0.2])
    P = x.shape[-1]
    assert P == 11
    lo, hi = np.full(P, -np.inf), np.full(P, np.inf)
    c, w = wl.params[:, :5].mean(axis=0), 0.4 * np.ptp(wl.params[:, :5], axis=0)
    lo[:5], hi[:5] = c - w, c + w
    ll = lambda rows: (orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, rows, wl.f_edges, h0e, summ)["logL"], {})
    logL = ll(x.reshape(n_t * n_w, -1))[0].reshape(n_t, n_w).copy()
    gx, gl = dev(tc, x), dev(tc, logL)
    acc_g = tc.zeros(n_t, dtype=tc.int64, device="cuda")
    n_acc = sm.run(x, logL, betas, lo, hi, 5, 2.0, 333, 0, 8, ll)
    ctx.pt_run(gx, gl, None, None, dev(tc, betas), dev(tc, lo), dev(tc, hi), 5, 333, 0, 8, n_accepted=acc_g)
    assert np.array_equal(gx.cpu().numpy(), x) and np.array_equal(acc_g.cpu().numpy(), n_acc) and n_acc.sum() > 50
    ctx.destroy()


# --------------------------------------------------------------------------- t_shift outside the spline (reading R32)
@pytest.mark.parametrize("n_m,n_c,n_w", [(1, 2, 97), (3, 2, 50), (1, 3, 40)])
def test_t_shift_array_entry_points(orc, torch_cuda, n_m, n_c, n_w):
    """Psi_m(f) = spline_m(f) + 2 pi f t_shift with t_shift ~ 1e5-1e6 s (1e3-1e5 rad across the band, several quarter
    cycles per bin) on ll_full_batch, _tf, _pw and ll_het_batch, against the oracle's long-double sum of the two terms."""
    from oracle import per_walker as pw
    from paper_2111_01064_b200 import binding
    tc = torch_cuda
    rng = np.random.default_rng(3200 + 10 * n_m + n_c)
    grid = wlm.make_grid(2.0 ** 17)
    f = grid.freqs()
    f_nodes = wlm.geomspace_exact(wlm.F_LO, wlm.F_HI, 80)
    W = _weights(rng, grid, n_c, n_c == 3)
    amp, ph = rand_smooth_nodes(rng, n_w, n_m, f_nodes)
    tf = unit_tf(rng, n_w, n_m, n_c)
    d = _noise(rng, grid, n_c)
    t_shift = rng.uniform(0.3, 0.9, n_w) * 2.0 ** 17 * rng.choice([-1.0, 1.0], n_w)
    t_shift[0] = 0.0
    lo = rng.uniform(0.5e-4, 5e-3, n_w)
    band = np.stack([lo, lo * rng.uniform(1.0, 40.0, n_w)], axis=1)
    ctx = binding.Context(n_modes=n_m, n_channels=n_c)
    ctx.set_data(grid.n_f, grid.k_min, grid.df, dev(tc, d), dev(tc, W))
    args = (dev(tc, amp), dev(tc, ph), dev(tc, tf), dev(tc, band))
    got = ctx.full_batch(f_nodes, *args, t_shift=dev(tc, t_shift))
    ref = orc.full_batch(f_nodes, amp, ph, tf, band, grid.k_min, grid.df, d, W, t_shift=t_shift)
    check_triplet(got, ref, "t_shift full_batch")
    plain = ctx.full_batch(f_nodes, *args)
    assert float((plain[1] - got[1]).abs().max()) > 1e-3 * float(got[2].abs().max()) ** 0.5      # the term does something
    assert abs(float(plain[1][0] - got[1][0])) <= 1e-9 * max(1.0, abs(float(got[1][0])))          # ... and nothing at 0
    tfn = _smooth_tf_nodes(rng, n_w, n_m, f_nodes, n_c)
    got = ctx.full_batch_tf(f_nodes, dev(tc, amp), dev(tc, ph), dev(tc, tfn), dev(tc, band), t_shift=dev(tc, t_shift))
    ref = orc.full_batch_tf(f_nodes, amp, ph, tfn, band, grid.k_min, grid.df, d, W, t_shift=t_shift)
    check_triplet(got, ref, "t_shift full_batch_tf")
    x = np.stack([np.geomspace(f[0] * rng.uniform(0.8, 1.5), f[-1] * rng.uniform(0.4, 1.1), 64) for _ in range(n_w)])
    ampw, phw = (np.stack([rand_smooth_nodes(rng, 1, n_m, x[w])[k][0] for w in range(n_w)]) for k in (0, 1))
    got = ctx.full_batch_pw(dev(tc, x), dev(tc, ampw), dev(tc, phw), dev(tc, tf), dev(tc, band), t_shift=dev(tc, t_shift))
    ref = pw.full_batch_pw(x, ampw, phw, tf, band, grid.k_min, grid.df, d, W, t_shift=t_shift)
    check_triplet(got, ref, "t_shift full_batch_pw")
    # heterodyne array entry
    e = wlm.geomspace_exact(f[3], f[-5] * 0.31, 33)
    h0 = rng.standard_normal((n_c, grid.n_f, 2)) * np.abs(d).mean() + np.abs(d).mean() * 3
    h0e = rng.standard_normal((n_c, len(e), 2)) + 3.0
    summ = orc.het_prepare(grid.k_min, grid.df, d, W, h0, e)
    amp_e = rng.uniform(0.5, 2.0, (n_w, n_m, len(e)))
    ph_e = rng.uniform(-2e4, 2e4, (n_w, n_m, len(e)))
    ctx.het_prepare(e, dev(tc, h0), dev(tc, h0e))
    got = ctx.het_batch(dev(tc, amp_e), dev(tc, ph_e), dev(tc, tf), t_shift=dev(tc, t_shift))
    check_triplet(got, orc.het_batch(e, amp_e, ph_e, tf, h0e, summ, t_shift=t_shift), "t_shift het_batch")
    ctx.destroy()


@pytest.mark.parametrize("index", [0, 3])
def test_standin_split_tc(orc, torch_cuda, index):
    """ll_standin_split_tc: the stand-in's linear term 2 pi f t_c kept outside the spline (one mode and six modes).
    Against the oracle doing the same, and — same template, reading R32 — against the oracle splining the full phase."""
    tc = torch_cuda
    if index == 0:
        wl = wlm.make_workload(0)
    else:
        wl = wlm.make_workload(3, n_w=48, t_obs=2.0 ** 16, n_knots=24)
        wl.path = "full"
        wl.f_nodes = wlm.geomspace_exact(wlm.F_LO, wlm.F_HI, 200)
    d, run = oracle_setup_full(orc, wl)
    g = wl.grid
    ctx = make_ctx(wl)
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    ctx.standin_split_tc(True)
    got = ctx.full_batch_standin(wl.f_nodes, dev(tc, wl.params))
    ref_split = orc.full_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params, wl.f_nodes, g.k_min, g.df, g.n_f, d, wl.W,
                                       split_tc=True)
    check_triplet(got, ref_split, f"split t_c cfg{index}")
    check_triplet(got, run(wl.params, d), f"split t_c vs the full-phase spline cfg{index}")
    # the node arrays of the caller layout follow the switch: phase without the linear term
    f = g.freqs()
    am, ph, _, _ = orc.standin_nodes(wl.params[:9], wl.modes_m, wl.c_lm, wl.kappa, wl.f_nodes, f[0], f[-1], split_tc=True)
    g_am, g_ph = (x.cpu().numpy() for x in ctx.standin_nodes(wl.f_nodes, dev(tc, wl.params[:9])))
    np.testing.assert_allclose(g_ph, ph, rtol=1e-13, atol=1e-9)
    h = ctx.full_template_standin(wl.f_nodes, wl.params[3]).cpu().numpy()
    href = run(wl.params[3][None], None, True)["h"]
    assert np.abs(h - href).max() <= 1e-8 * np.abs(href).max()
    ctx.standin_split_tc(False)
    check_triplet(ctx.full_batch_standin(wl.f_nodes, dev(tc, wl.params)), run(wl.params, d), "switch off again")
    ctx.destroy()


def test_unsupported_layouts_are_errors(torch_cuda):
    from paper_2111_01064_b200 import binding
    tc = torch_cuda
    for bad in (1, 4):
        with pytest.raises(binding.LLError) as ei:
            binding.Context(n_modes=1, n_channels=bad)
        assert ei.value.code == binding.LL_ERR_UNSUPPORTED
    ctx = binding.Context(n_modes=1, n_channels=3, precision=binding.LL_PREC_FP32_ACC)
    with pytest.raises(binding.LLError) as ei:
        ctx.set_data(100, 10, 1e-5, tc.zeros((3, 100, 2), dtype=tc.float64, device="cuda"),
                     tc.ones((3, 100), dtype=tc.float64, device="cuda"))
    assert ei.value.code == binding.LL_ERR_UNSUPPORTED
    ctx.destroy()
    ctx = binding.Context(n_modes=1, n_channels=3)
    with pytest.raises(ValueError):
        ctx.set_data(100, 10, 1e-5, tc.zeros((2, 100, 2), dtype=tc.float64, device="cuda"),
                     tc.ones(100, dtype=tc.float64, device="cuda"))
    with pytest.raises(ValueError):
        ctx.set_data(100, 10, 1e-5, tc.zeros((3, 100, 2), dtype=tc.float64, device="cuda"),
                     tc.ones((2, 100), dtype=tc.float64, device="cuda"))
    ctx.destroy()


def test_memory_checks(torch_cuda):
    """every kernel family once (both channel counts, small and large routes, the sampler in both forms), then the guard
    bands behind every internal device buffer must be intact (ll_debug_check); outputs must be finite"""
    from paper_2111_01064_b200 import sanitize_smoke
    assert sanitize_smoke.main() == 0
