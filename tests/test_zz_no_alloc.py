"""ll_pt_stretch_half_het_static (include/ll.h): the sampler's half update with its scratch in the library's
file-scope device array, for callers that must not allocate.  Checked against the existing path,
ll_pt_stretch_half_het, on two calls in a row (half 0, then half 1) from the same starting state.

This file sorts last on purpose (the suite runs with `pytest -x`): a failure here hides no other test.  It builds
its own small heterodyne set-up, so it passes alone in a fresh process and after the other tests alike; the static
calls run on a context that has never taken a sampler step (its lazily grown sampler buffers do not exist)."""
import numpy as np
import pytest

from paper_2111_01064_b200 import workloads as wlm
from helpers import check_triplet, dev, make_ctx, oracle_setup_het

pytestmark = pytest.mark.gpu


def _prepared_ctx(wl, tc, d, h0, h0e):
    ctx = make_ctx(wl)
    g = wl.grid
    ctx.set_data(g.n_f, g.k_min, g.df, dev(tc, d), dev(tc, wl.W))
    ctx.het_prepare(wl.f_edges, dev(tc, h0), dev(tc, h0e))
    return ctx


def test_static_scratch_half_update_matches_existing_path(orc, torch_cuda):
    tc = torch_cuda
    from paper_2111_01064_b200 import binding
    wl = wlm.make_workload(1, n_w=300, t_obs=2.0 ** 18, n_knots=37)
    d, h0, h0e, _ = oracle_setup_het(orc, wl)
    ctx_ref = _prepared_ctx(wl, tc, d, h0, h0e)      # takes the existing path
    ctx_sta = _prepared_ctx(wl, tc, d, h0, h0e)      # takes the static-scratch path, and nothing else of the sampler

    n_t, n_w = 3, 64
    x0 = wl.params[:n_t * n_w].reshape(n_t, n_w, -1).copy()
    x0[:, :, 5:] = wl.inj[5:]                         # frozen coordinates
    P = x0.shape[-1]
    lo, hi = np.full(P, -np.inf), np.full(P, np.inf)
    c, w = wl.params[:, :5].mean(axis=0), 0.35 * np.ptp(wl.params[:, :5], axis=0)
    lo[:5], hi[:5] = c - w, c + w                     # tight enough that some proposals leave the box
    gb, glo, ghi = dev(tc, np.array([1.0, 0.3, 0.05])), dev(tc, lo), dev(tc, hi)
    first = ctx_ref.het_batch_standin(dev(tc, x0.reshape(n_t * n_w, P)))

    def state():
        return [dev(tc, x0)] + [v.reshape(n_t, n_w).clone() for v in first]

    ref, sta = state(), state()
    acc_ref = tc.full((n_t, n_w // 2), -1, dtype=tc.int32, device="cuda")
    acc_sta = tc.full((n_t, n_w // 2), -1, dtype=tc.int32, device="cuda")
    rng = np.random.default_rng(2111)
    n_acc = 0
    for half in (0, 1):                               # two calls in a row: the second finds the first one's scratch
        u = [dev(tc, v) for v in rng.random((3, n_t, n_w // 2))]
        ctx_ref.pt_stretch_half(half, *ref, gb, glo, ghi, 5, *u, accepted=acc_ref)
        ctx_sta.pt_stretch_half_static(half, *sta, gb, glo, ghi, 5, *u, accepted=acc_sta)
        tc.cuda.synchronize()
        assert tc.equal(acc_sta, acc_ref), f"accept decisions, half {half}"
        assert tc.equal(sta[0], ref[0]), f"positions, half {half}"
        check_triplet([v.reshape(-1) for v in sta[1:]],
                      {k: v.reshape(-1).cpu().numpy() for k, v in zip(("logL", "d_h", "h_h"), ref[1:])},
                      f"static scratch, half {half}")
        n_acc += int(acc_ref.sum())
    assert 10 < n_acc < n_t * n_w                     # the step did something, and not everything
    assert not tc.equal(ref[0], dev(tc, x0))

    # beyond the array: refused with the limit named, nothing launched, the state untouched
    big_t, big_w = 1, 2 * 20000                       # 20 000 proposals of 9 parameters: 2.16 MB > LL_STATIC_SCRATCH_BYTES
    assert (big_w // 2) * (P + 4.5) * 8 > binding.LL_STATIC_SCRATCH_BYTES
    xb = tc.zeros((big_t, big_w, P), dtype=tc.float64, device="cuda")
    lb = [tc.zeros((big_t, big_w), dtype=tc.float64, device="cuda") for _ in range(3)]
    ub = [tc.full((big_t, big_w // 2), 0.5, dtype=tc.float64, device="cuda") for _ in range(3)]
    launches = ctx_sta.kernel_launches()
    with pytest.raises(binding.LLError, match="LL_STATIC_SCRATCH_BYTES"):
        ctx_sta.pt_stretch_half_static(0, xb, *lb, gb[:1].contiguous(), glo, ghi, 5, *ub)
    assert ctx_sta.kernel_launches() == launches
    # and the array still serves the next call that fits
    u = [dev(tc, v) for v in rng.random((3, n_t, n_w // 2))]
    ctx_ref.pt_stretch_half(0, *ref, gb, glo, ghi, 5, *u, accepted=acc_ref)
    ctx_sta.pt_stretch_half_static(0, *sta, gb, glo, ghi, 5, *u, accepted=acc_sta)
    assert tc.equal(acc_sta, acc_ref) and tc.equal(sta[0], ref[0])
    assert ctx_sta.debug_check() == 0 and ctx_ref.debug_check() == 0
    ctx_ref.destroy()
    ctx_sta.destroy()
