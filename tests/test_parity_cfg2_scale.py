"""GPU parity tests (-m gpu) at BASELINE.json config 2's FULL size for every full-grid kernel bench.py times there
(`per_config.cfg2`, `cfg2_tf`, `cfg2_pw`, `cfg2_hm6`, `module1_iteration`): the one-year grid (1 574 725 bins), 1024
nodes, LISA-scale phases (up to ~1e7 rad, several quarter cycles per bin), the launch configuration of the bench, and
the oracle recomputing sampled walkers one by one.  Each of those kernels carries its own copy of the rotation
recurrence (ll_kernels.cuh), so each needs its own test at this scale.

Tolerance (BASELINE.json north_star): |delta log L| <= 1e-6 max(1, |log L|), d_h and h_h separately
at 1e-6 max(1, |h_h|).  Inputs: the seeded config-2 workload (workloads.py), completed with the oracle (helpers.py);
node arrays for the array entry points come from a numpy generator in this file, never from the CUDA path.
"""
import numpy as np
import pytest

from paper_2111_01064_b200 import workloads as wlm
from helpers import check_triplet, dev, make_ctx, oracle_setup_full

pytestmark = pytest.mark.gpu


def _np_triplet(got, idx):
    import torch
    return [torch.as_tensor(x[idx]) for x in got]


def sample_walkers(n_w, fis, extra=(), stride=None, wb=128):
    """walker 0, min / max f_ISCO (shortest / longest band), walker-block boundaries of the launch, every `stride`-th"""
    s = {0, 1, int(fis.argmin()), int(fis.argmax()), wb - 1, wb, n_w - wb - 1, n_w - wb, n_w - 1} | set(extra)
    if stride:
        s |= set(range(stride // 3, n_w, stride))
    return np.array(sorted(i for i in s if 0 <= i < n_w))


def lisa_node_arrays(params, x, kappa=wlm.KAPPA):
    """INPUT GENERATOR for the array entry points (ll_full_batch / _tf / _pw take whatever amplitude and phase they are
    given): smooth node arrays with the magnitude and the phase scale of a LISA massive-black-hole binary — amplitude
    ~ f^(-7/6)/D rolled off above a walker-dependent frequency, phase 2 pi f t_c + K f^(-5/3) + const reaching ~1e7
    rad — at the nodes x [n_w][n_nodes] (or [n_nodes]).  numpy float64; both the oracle and the library get these arrays."""
    x = np.broadcast_to(np.asarray(x, dtype=np.float64), (params.shape[0], np.shape(x)[-1]))
    mc, q, tc, phic, inv_d = (params[:, k][:, None] for k in range(5))
    eta = q / (1.0 + q) ** 2
    mtot = mc * eta ** -0.6
    f_roll = 6.0 ** -1.5 / (np.pi * mtot)
    s = np.clip((1.0 + kappa - x / f_roll) / kappa, 0.0, 1.0)
    amp = x ** (-7.0 / 6.0) * inv_d * s ** 3 * (10.0 - 15.0 * s + 6.0 * s * s)
    phase = 2.0 * np.pi * x * tc - phic - 0.25 * np.pi + 3.0 / (128.0 * eta) * (np.pi * mtot * x) ** (-5.0 / 3.0)
    band_top = np.minimum((1.0 + kappa) * f_roll[:, 0], wlm.F_HI)
    return np.ascontiguousarray(amp[:, None, :]), np.ascontiguousarray(phase[:, None, :]), band_top


@pytest.fixture(scope="module")
def cfg2(orc, torch_cuda):
    wl = wlm.make_workload(2)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(torch_cuda, d), dev(torch_cuda, wl.W))
    fis = np.array([orc.standin_fisco(p) for p in wl.params])
    yield wl, d, run, ctx, fis
    ctx.destroy()


def test_cfg2_full_size_128_walkers(cfg2, torch_cuda):
    """k_full_fused<1> (bench headline, per_config.cfg2): >= 128 sampled walkers of the full 16384-walker batch
    against the oracle (BASELINE.md §3 planned a 512-walker subset; the oracle does ~38 walkers/s on 16 cores)."""
    wl, d, run, ctx, fis = cfg2
    got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))]
    sample = sample_walkers(wl.n_w, fis, stride=128)
    assert len(sample) >= 128
    ref = run(wl.params[sample], d)
    check_triplet(_np_triplet(got, sample), ref, "cfg2 full size, 128+ walkers")


@pytest.mark.parametrize("n_small", [37, 160, 320, 1024, 2048])
def test_module1_sized_batches_against_oracle(cfg2, torch_cuda, n_small):
    """Module-1 sized batches on the one-year grid (80 walkers x 4 temperatures; a half update is 160
    proposals, a whole population 320): the small-batch route (per_config.module1_iteration) against the ORACLE, not
    only against the large-batch route.  1024: the largest batch of the small-batch route (32 groups); 2048: the
    large-batch route just above it (per_config.cfg2_batch_sizes)."""
    wl, d, run, ctx, fis = cfg2
    rng = np.random.default_rng(194 + n_small)
    idx = rng.choice(wl.n_w, n_small, replace=False)
    idx[0] = 0                                              # the injection: log L ~ -n_f (noise), <d|h> = 2.5e5
    params = wl.params[idx]
    got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, params))]
    sample = np.arange(n_small) if n_small <= 40 else np.unique(np.r_[0, 31, 32, n_small - 1, rng.integers(0, n_small, 36)])
    ref = run(params[sample], d)
    check_triplet(_np_triplet(got, sample), ref, f"module-1 sized batch of {n_small}")


def _smooth_tf_at_nodes(params, f_nodes, n_c=2):
    """smooth complex T^c(f_j) per walker (the response's formula is in the paper's ref. [44], not in PAPER.md):
    the walker's constant factor times (1 + 0.2 x) e^{2 i x}(1 + 0.1 sin(5 x + phi_c)), x = log-frequency in [0, 1]"""
    x = np.log(f_nodes / f_nodes[0]) / np.log(f_nodes[-1] / f_nodes[0])
    n_w = params.shape[0]
    t0 = params[:, 5:5 + 2 * n_c].reshape(n_w, 1, n_c, 1, 2)
    mod = (1.0 + 0.2 * x)[None, :] * (1.0 + 0.1 * np.sin(5.0 * x[None, :] + params[:, 3:4]))
    cr, ci = (mod * np.cos(2.0 * x))[:, None, None, :], (mod * np.sin(2.0 * x))[:, None, None, :]
    out = np.stack([t0[..., 0] * cr - t0[..., 1] * ci, t0[..., 0] * ci + t0[..., 1] * cr], axis=-1)
    return np.ascontiguousarray(out)


def test_cfg2_tf_full_size_sampled(cfg2, orc, torch_cuda):
    """k_full_fused_tf<1> (per_config.cfg2_tf): frequency-dependent transfer function (Eq. 8-9) on the full
    16384-walker batch, one-year grid, LISA-scale phases, the walkers' own bands; 18 sampled walkers vs oracle.full_batch_tf."""
    wl, d, run, ctx, fis = cfg2
    amp, ph, top = lisa_node_arrays(wl.params, wl.f_nodes)
    tfn = _smooth_tf_at_nodes(wl.params, wl.f_nodes)
    g = wl.grid
    band = np.ascontiguousarray(np.stack([np.full(wl.n_w, g.k_min * g.df), top], axis=1))
    tc = torch_cuda
    got = [x.cpu().numpy() for x in ctx.full_batch_tf(wl.f_nodes, dev(tc, amp), dev(tc, ph), dev(tc, tfn), dev(tc, band))]
    sample = sample_walkers(wl.n_w, fis, stride=2048)
    assert len(sample) >= 16
    ref = orc.full_batch_tf(wl.f_nodes, amp[sample], ph[sample], tfn[sample], band[sample], g.k_min, g.df, d, wl.W)
    assert np.abs(ph).max() > 5e6                          # LISA-scale phases (2 pi f t_c at 0.05 Hz, t_c ~ 0.9 yr)
    check_triplet(_np_triplet(got, sample), ref, "cfg2 tf sampled")
    assert np.all(np.isfinite(got[0]))


def test_cfg2_pw_full_size_sampled(cfg2, orc, torch_cuda):
    """k_full_fused_pw<1> (per_config.cfg2_pw): per-walker node grids on the full 16384-walker batch.  Even walkers
    carry a copy of the shared 1024 nodes, odd walkers 1024 log-spaced nodes over their OWN span (starting above the
    grid's first bin, ending near their band top), so lanes of one warp sit in different intervals of different
    widths; 20 sampled walkers vs oracle.per_walker.full_batch_pw."""
    from oracle import per_walker as pw
    wl, d, run, ctx, fis = cfg2
    g = wl.grid
    rng = np.random.default_rng(30)
    _, _, top = lisa_node_arrays(wl.params, wl.f_nodes)
    x = np.tile(wl.f_nodes, (wl.n_w, 1))
    odd = np.arange(1, wl.n_w, 2)
    lo = wlm.F_LO * rng.uniform(1.0, 3.0, len(odd))
    hi = np.minimum(top[odd] * rng.uniform(0.7, 1.1, len(odd)), wlm.F_HI)
    t = np.linspace(0.0, 1.0, len(wl.f_nodes))
    x[odd] = np.exp(np.log(lo)[:, None] + (np.log(hi) - np.log(lo))[:, None] * t[None, :])
    x[odd, 0], x[odd, -1] = lo, hi
    amp, ph, _ = lisa_node_arrays(wl.params, x)
    tf = np.ascontiguousarray(wl.params[:, 5:9].reshape(wl.n_w, 1, 2, 2))
    band = np.ascontiguousarray(np.stack([np.full(wl.n_w, g.k_min * g.df), top], axis=1))
    tc = torch_cuda
    got = [v.cpu().numpy() for v in ctx.full_batch_pw(dev(tc, x), dev(tc, amp), dev(tc, ph), dev(tc, tf), dev(tc, band))]
    sample = sample_walkers(wl.n_w, fis, extra=(2, 3, 4097, 4098), stride=2048)
    assert len(sample) >= 16 and (sample % 2 == 1).sum() >= 6 and (sample % 2 == 0).sum() >= 6
    ref = pw.full_batch_pw(x[sample], amp[sample], ph[sample], tf[sample], band[sample], g.k_min, g.df, d, wl.W)
    check_triplet(_np_triplet(got, sample), ref, "cfg2 per-walker nodes sampled")
    assert np.all(np.isfinite(got[0]))


@pytest.mark.parametrize("n_m,n_w", [(6, 2048), (3, 2048), (6, 1000), (6, 500), (6, 160), (3, 45)])
def test_cfg2_hm6_full_size_sampled(orc, torch_cuda, n_m, n_w):
    """k_full_fused_hm<6 | 3, 2, true> (per_config.cfg2_hm6: every mode by its own rotation recurrence): config 3's six
    modes (or the first three) through the FULL-GRID path on config 2's one-year grid and 1024 nodes, 2048 prior-draw
    walkers (the bench's batch); data = walker 0's template + noise; 16 sampled walkers vs the oracle; with three modes
    also with 2 pi f t_c kept outside the splines (t_shift in every mode's phase cubic); 1000 walkers: the smallest batches
    that take the large route (from 960 walkers on); 500, 160 and 45 walkers: the kernel's item form on the small-batch route."""
    wl6, wl2 = wlm.make_workload(3, n_w=8), wlm.make_workload(2, n_w=n_w)
    wl6.n_m, wl6.modes_l, wl6.modes_m, wl6.c_lm = n_m, wl6.modes_l[:n_m], wl6.modes_m[:n_m], wl6.c_lm[:n_m]
    rng = np.random.default_rng(wlm.SEED_BASE + 232)
    params = np.empty((n_w, 5 + 4 * wl6.n_m))
    params[:, :5] = wl2.params[:, :5]
    ang = rng.uniform(0, 2 * np.pi, (n_w, 2 * wl6.n_m))
    params[:, 5::2], params[:, 6::2] = np.cos(ang), np.sin(ang)
    g = wl2.grid
    run = lambda p, dd, t=False: orc.full_batch_standin(wl6.modes_m, wl6.c_lm, wl6.kappa, p, wl2.f_nodes, g.k_min, g.df,
                                                        g.n_f, dd, wl2.W, want_template=t)
    hh = run(params[:1], None)["h_h"][0]
    params[:, 4] *= wlm.SNR_TARGET / np.sqrt(hh)            # walker 0 at SNR 500 (reading R18)
    d = run(params[:1], None, True)["h"] + wl2.noise
    from paper_2111_01064_b200 import binding
    ctx = binding.Context(n_modes=wl6.n_m)
    ctx.standin_config(wl6.modes_l, wl6.modes_m, wl6.c_lm, wl6.kappa)
    tc = torch_cuda
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl2.W))
    got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl2.f_nodes, dev(tc, params))]
    fis = np.array([orc.standin_fisco(p) for p in params])
    sample = sample_walkers(n_w, fis, stride=256 if n_w > 1000 else (40 if n_w > 300 else (10 if n_w > 100 else 3)), wb=64)
    assert len(sample) >= min(16, n_w // 3)
    ref = run(params[sample], d)
    check_triplet(_np_triplet(got, sample), ref, f"cfg2 {n_m} modes sampled")
    assert abs(np.sqrt(got[2][0]) - 500.0) < 1e-3
    if n_m == 3:
        ctx.standin_split_tc(True)
        got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl2.f_nodes, dev(tc, params))]
        ref = orc.full_batch_standin(wl6.modes_m, wl6.c_lm, wl6.kappa, params[sample], wl2.f_nodes, g.k_min, g.df, g.n_f, d,
                                     wl2.W, split_tc=True)
        check_triplet(_np_triplet(got, sample), ref, "cfg2 3 modes, t_c outside the spline")
    ctx.destroy()


def test_cfg2_three_channels_full_size_sampled(orc, torch_cuda):
    """k_full_fused<1, 3, false> (per_config.cfg2_nc3): config 2 with three channels (A, E, T; the T channel with its own
    PSD) at full size, 16 384 walkers with 11-double rows; 18 sampled walkers vs the oracle."""
    wl = wlm.make_workload(2, n_c=3)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    tc = torch_cuda
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(tc, wl.params))]
    fis = np.array([orc.standin_fisco(p) for p in wl.params])
    sample = sample_walkers(wl.n_w, fis, stride=2048)
    assert len(sample) >= 16
    ref = run(wl.params[sample], d)
    check_triplet(_np_triplet(got, sample), ref, "cfg2 three channels sampled")
    assert np.all(np.isfinite(got[0])) and abs(np.sqrt(got[2][0]) - 500.0) < 1e-3
    ctx.destroy()


def test_cfg2_split_tc_full_size_sampled(cfg2, orc, torch_cuda):
    """per_config.cfg2_split_tc: the stand-in's linear term 2 pi f t_c (up to ~9e6 rad) kept outside the spline as
    t_shift (reading R32) on the full config-2 batch; sampled walkers vs the oracle doing the same (long-double sum of the
    two phase terms), and vs the oracle splining the full phase (the same template up to rounding)."""
    wl, d, run, ctx, fis = cfg2
    g = wl.grid
    ctx.standin_split_tc(True)
    try:
        got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params))]
    finally:
        ctx.standin_split_tc(False)
    sample = sample_walkers(wl.n_w, fis, stride=1024)
    ref = orc.full_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params[sample], wl.f_nodes, g.k_min, g.df, g.n_f, d, wl.W,
                                 split_tc=True)
    check_triplet(_np_triplet(got, sample), ref, "cfg2 split t_c sampled")
    ref_full = run(wl.params[sample], d)
    check_triplet(_np_triplet(got, sample), ref_full, "cfg2 split t_c vs the full-phase spline")
    # what the split buys: distance of <d|h> from the oracle, split vs full-phase (reported in DESIGN.md §6)
    plain = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(torch_cuda, wl.params[sample]))]
    e_split = np.abs(got[1][sample] - ref["d_h"]).max()
    e_plain = np.abs(plain[1] - ref_full["d_h"]).max()
    print(f"max |d_h - oracle|: split t_c {e_split:.3e}, full-phase spline {e_plain:.3e}; "
          f"oracle split vs oracle full {np.abs(ref['d_h'] - ref_full['d_h']).max():.3e}")


# ------------------------------------------------------------------------------------------------------------------
# The small-batch route's LANES ITEMS (ll_kernels.cuh: a group's range above its lowest band top goes to sub-groups of 16
# walkers x 2 bin phases) exist only where the spline intervals are long, i.e. on this grid; the tests above cover them for
# the stand-in entry point with two channels.  The other ways into the same kernel, at Module-1 size:
def test_small_batch_three_channels_against_oracle(orc, torch_cuda):
    """160 walkers, three channels with per-channel PSDs (k_full_fused<1, 3, false, SMALL>: the lanes items' <h|h> from the
    moments of every weight row), one-year grid, against the oracle."""
    wl = wlm.make_workload(2, n_c=3)
    d, run = oracle_setup_full(orc, wl)
    ctx = make_ctx(wl)
    g = wl.grid
    tc = torch_cuda
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    rng = np.random.default_rng(1943)
    idx = rng.choice(wl.n_w, 160, replace=False)
    idx[0] = 0
    params = wl.params[idx]
    got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(tc, params))]
    sample = np.unique(np.r_[0, 15, 16, 31, 32, 159, rng.integers(0, 160, 18)])
    check_triplet(_np_triplet(got, sample), run(params[sample], d), "three channels, 160 walkers")
    ctx.destroy()


def test_small_batch_split_tc_and_arrays_against_oracle(cfg2, orc, torch_cuda):
    """160 walkers through (i) the stand-in entry point with 2 pi f t_c kept outside the spline (t_shift folded into the
    lanes items' phase cubic) and (ii) the array entry point ll_full_batch with per-walker bands and t_shift (planner, node
    transposition and spline as separate launches; bands with different bottoms), both against the oracle."""
    wl, d, run, ctx, fis = cfg2
    g = wl.grid
    tc = torch_cuda
    rng = np.random.default_rng(1944)
    idx = rng.choice(wl.n_w, 160, replace=False)
    params = wl.params[idx]
    sample = np.unique(np.r_[0, 15, 16, 31, 32, 159, rng.integers(0, 160, 14)])
    # (i)
    ctx.standin_split_tc(True)
    try:
        got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(tc, params))]
    finally:
        ctx.standin_split_tc(False)
    ref = orc.full_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, params[sample], wl.f_nodes, g.k_min, g.df, g.n_f, d, wl.W,
                                 split_tc=True)
    check_triplet(_np_triplet(got, sample), ref, "split t_c, 160 walkers")
    # (ii) numpy-generated node arrays, the linear term as t_shift, bands starting at different bins
    amp, phase, top = lisa_node_arrays(params, wl.f_nodes)
    phase = phase - 2.0 * np.pi * wl.f_nodes[None, None, :] * params[:, 2][:, None, None]
    band = np.stack([wlm.F_LO * (1.0 + 3.0 * rng.random(160)), top], axis=1)
    tf = np.ascontiguousarray(params[:, 5:9].reshape(160, 1, 2, 2))
    ts = np.ascontiguousarray(params[:, 2])
    got = [x.cpu().numpy() for x in ctx.full_batch(wl.f_nodes, dev(tc, amp), dev(tc, phase), dev(tc, tf), dev(tc, band),
                                                   t_shift=dev(tc, ts))]
    ref = orc.full_batch(wl.f_nodes, amp[sample], phase[sample], tf[sample], band[sample], g.k_min, g.df, d, wl.W,
                         t_shift=ts[sample])
    check_triplet(_np_triplet(got, sample), ref, "array entry point, 160 walkers")


@pytest.mark.parametrize("n", [1, 17, 33, 49, 257, 513])
def test_small_batch_odd_sizes_and_bands(cfg2, orc, torch_cuda, n):
    """The planner's corner cases on the one-year grid: batch sizes that leave sub-groups and groups partly empty, walkers
    with identical bands (no ragged part: n divisible by 3), and — through the array entry point — bands that are empty,
    a few bins wide, or start high on the grid; 513 walkers take the separate-launch set-up.  Sampled walkers vs the oracle;
    the guard bands of every internal buffer afterwards."""
    wl, d, run, ctx, fis = cfg2
    g = wl.grid
    tc = torch_cuda
    rng = np.random.default_rng(3000 + n)
    p = wl.params[rng.choice(wl.n_w, n, replace=False)].copy()
    if n % 3 == 0:
        p[:, 0], p[:, 1] = p[0, 0], p[0, 1]
    s = np.unique(np.r_[0, n - 1, rng.integers(0, n, 8)])
    got = [x.cpu().numpy() for x in ctx.full_batch_standin(wl.f_nodes, dev(tc, p))]
    check_triplet(_np_triplet(got, s), run(p[s], d), f"stand-in entry, {n} walkers")
    amp, phase, top = lisa_node_arrays(p, wl.f_nodes)
    lo = wlm.F_LO * (1.0 + 20.0 * rng.random(n) ** 3)
    hi = np.where(rng.random(n) < 0.1, 0.5 * lo, np.minimum(top, lo * (1.0 + 50.0 * rng.random(n))))  # 10 % empty bands
    if n >= 4:
        hi[1] = lo[1] * 1.0001          # a handful of bins
        lo[2], hi[2] = 0.03, 0.05       # only the top of the grid
    band = np.stack([lo, hi], axis=1)
    tf = np.ascontiguousarray(p[:, 5:9].reshape(n, 1, 2, 2))
    got = [x.cpu().numpy() for x in ctx.full_batch(wl.f_nodes, dev(tc, amp), dev(tc, phase), dev(tc, tf), dev(tc, band))]
    ref = orc.full_batch(wl.f_nodes, amp[s], phase[s], tf[s], band[s], g.k_min, g.df, d, wl.W)
    check_triplet(_np_triplet(got, s), ref, f"array entry, {n} walkers")
    assert ctx.debug_check() == 0


def test_multi_mode_arrays_with_scattered_bands(orc, torch_cuda):
    """k_full_fused_hm through the array entry point: 1100 walkers, three modes, bands scattered over the grid (narrow, low,
    high, empty), so that the union of a warp's bands has holes and the kernel's recurrence has to restart where the bins
    stop being contiguous; sampled walkers vs the oracle."""
    n_w, n_m = 1100, 3
    wl = wlm.make_workload(2, n_w=n_w)
    g = wl.grid
    rng = np.random.default_rng(2320)
    a1, p1, top = lisa_node_arrays(wl.params, wl.f_nodes)
    scale = np.array([1.0, 0.4, 0.25])[None, :, None]
    amp = np.ascontiguousarray(a1 * scale)
    phase = np.ascontiguousarray(p1 * np.array([1.0, 0.5, 1.5])[None, :, None])
    ang = rng.uniform(0, 2 * np.pi, (n_w, n_m, 2))
    tf = np.ascontiguousarray(np.stack([np.cos(ang), np.sin(ang)], axis=-1))
    lo = wlm.F_LO * (1.0 + 200.0 * rng.random(n_w) ** 2)
    hi = np.where(rng.random(n_w) < 0.05, 0.5 * lo, np.minimum(0.05, lo * (1.0 + 0.5 * rng.random(n_w))))
    band = np.stack([lo, hi], axis=1)
    d = wl.noise
    from paper_2111_01064_b200 import binding
    ctx = binding.Context(n_modes=n_m)
    tc = torch_cuda
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    got = [x.cpu().numpy() for x in ctx.full_batch(wl.f_nodes, dev(tc, amp), dev(tc, phase), dev(tc, tf), dev(tc, band))]
    s_ = np.unique(np.r_[0, 127, 128, n_w - 1, rng.integers(0, n_w, 20)])
    ref = orc.full_batch(wl.f_nodes, amp[s_], phase[s_], tf[s_], band[s_], g.k_min, g.df, d, wl.W)
    check_triplet(_np_triplet(got, s_), ref, "three modes, scattered bands")
    assert ctx.debug_check() == 0
    ctx.destroy()


@pytest.mark.parametrize("n", [160, 333])
def test_small_batch_tf_against_oracle(cfg2, orc, torch_cuda, n):
    """The frequency-dependent transfer function (Eq. 8-9) at Module-1 size on the one-year grid: k_full_fused_tf in its
    small-batch form (one-warp blocks over the planner's cost-balanced group items), bands with different bottoms and a
    t_shift, against oracle.full_batch_tf."""
    wl, d, run, ctx, fis = cfg2
    g = wl.grid
    tc = torch_cuda
    rng = np.random.default_rng(8900 + n)
    p = wl.params[rng.choice(wl.n_w, n, replace=False)]
    amp, ph, top = lisa_node_arrays(p, wl.f_nodes)
    ph = ph - 2.0 * np.pi * wl.f_nodes[None, None, :] * p[:, 2][:, None, None]
    ts = np.ascontiguousarray(p[:, 2])
    tfn = _smooth_tf_at_nodes(p, wl.f_nodes)
    band = np.ascontiguousarray(np.stack([wlm.F_LO * (1.0 + 2.0 * rng.random(n)), top], axis=1))
    got = [x.cpu().numpy() for x in ctx.full_batch_tf(wl.f_nodes, dev(tc, amp), dev(tc, ph), dev(tc, tfn), dev(tc, band),
                                                      t_shift=dev(tc, ts))]
    s_ = np.unique(np.r_[0, 31, 32, n - 1, rng.integers(0, n, 12)])
    ref = orc.full_batch_tf(wl.f_nodes, amp[s_], ph[s_], tfn[s_], band[s_], g.k_min, g.df, d, wl.W, t_shift=ts[s_])
    check_triplet(_np_triplet(got, s_), ref, f"T(f), {n} walkers")
    assert ctx.debug_check() == 0


@pytest.mark.parametrize("n,bc", [(160, 0), (333, 1)])
def test_small_batch_pw_against_oracle(cfg2, orc, torch_cuda, n, bc):
    """Per-walker node grids at Module-1 size on the one-year grid: k_spline_pw_block (a block per four walkers of a system;
    elimination factors from a 16-row warm-up, dp and M by scans of affine maps) instead of the thread-per-system sweep, with
    the natural and the not-a-knot boundary condition; every second walker has 1024 log-spaced nodes over its own span."""
    from oracle import per_walker as pw
    from paper_2111_01064_b200 import binding
    wl, d, run, ctx0, fis = cfg2
    g = wl.grid
    tc = torch_cuda
    rng = np.random.default_rng(5100 + n)
    p = wl.params[rng.choice(wl.n_w, n, replace=False)]
    _, _, top = lisa_node_arrays(p, wl.f_nodes)
    x = np.tile(wl.f_nodes, (n, 1))
    odd = np.arange(1, n, 2)
    lo = wlm.F_LO * rng.uniform(1.0, 3.0, len(odd))
    hi = np.minimum(top[odd] * rng.uniform(0.7, 1.1, len(odd)), wlm.F_HI)
    t = np.linspace(0.0, 1.0, len(wl.f_nodes))
    x[odd] = np.exp(np.log(lo)[:, None] + (np.log(hi) - np.log(lo))[:, None] * t[None, :])
    x[odd, 0], x[odd, -1] = lo, hi
    amp, ph, _ = lisa_node_arrays(p, x)
    tf = np.ascontiguousarray(p[:, 5:9].reshape(n, 1, 2, 2))
    band = np.ascontiguousarray(np.stack([np.full(n, g.k_min * g.df), top], axis=1))
    ctx = binding.Context(n_modes=1, spline_bc=bc)
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    got = [v.cpu().numpy() for v in ctx.full_batch_pw(dev(tc, x), dev(tc, amp), dev(tc, ph), dev(tc, tf), dev(tc, band))]
    s_ = np.unique(np.r_[0, 1, 2, 3, n - 2, n - 1, rng.integers(0, n, 10)])
    orc.set_spline_bc(bc)
    try:
        ref = pw.full_batch_pw(x[s_], amp[s_], ph[s_], tf[s_], band[s_], g.k_min, g.df, d, wl.W)
    finally:
        orc.set_spline_bc(0)
    check_triplet(_np_triplet(got, s_), ref, f"per-walker nodes, {n} walkers, bc {bc}")
    assert ctx.debug_check() == 0
    ctx.destroy()


def test_small_batch_reruns_are_bit_identical(cfg2, torch_cuda):
    """Every way into the small-batch route on the one-year grid, called again and again with the same inputs: the same bits
    (the planner's tables, the per-block ranking of k_setup_small, the lanes items' butterflies and the tickets of the split F4
    must not let timing into the sums)."""
    wl, d, run, ctx, fis = cfg2
    tc = torch_cuda
    rng = np.random.default_rng(77)
    p = wl.params[rng.choice(wl.n_w, 160, replace=False)]
    amp, ph, top = lisa_node_arrays(p, wl.f_nodes)
    g = wl.grid
    band = dev(tc, np.stack([np.full(160, g.k_min * g.df), top], axis=1))
    tf = dev(tc, p[:, 5:9].reshape(160, 1, 2, 2))
    tfn = dev(tc, _smooth_tf_at_nodes(p, wl.f_nodes))
    xw = dev(tc, np.tile(wl.f_nodes, (160, 1)))
    gp, ga, gph = dev(tc, p), dev(tc, amp), dev(tc, ph)
    calls = {"stand-in": lambda: ctx.full_batch_standin(wl.f_nodes, gp),
             "arrays": lambda: ctx.full_batch(wl.f_nodes, ga, gph, tf, band),
             "T(f)": lambda: ctx.full_batch_tf(wl.f_nodes, ga, gph, tfn, band),
             "per-walker nodes": lambda: ctx.full_batch_pw(xw, ga, gph, tf, band)}
    for name, fn in calls.items():
        first = [v.clone() for v in fn()]
        for rep in range(8):
            again = fn()
            assert all(tc.equal(a, b) for a, b in zip(first, again)), f"{name}: rerun {rep} differs"
