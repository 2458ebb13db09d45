"""One small invocation of every kernel family of libll_b200.so, as a memory check (SURVEY.md §5 asks for
`compute-sanitizer` memcheck / racecheck; that tool is closed on this pool, see profiles/r02_memory_checks.md):

    python -m paper_2111_01064_b200.sanitize_smoke          (also: tests/test_parity_channels.py::test_memory_checks)

After every family the context's guard bands are read back (`ll_debug_check`: a canary band behind every internal
device buffer; an out-of-bounds store by any kernel shows up there).  Built with LL_NVCC_FLAGS=-DLL_POISON_STAGES the
fused kernels also overwrite every stage of the TMA ring with NaNs once they are done with it, so a read that beat its
bulk copy would turn the outputs into NaNs: the whole `-m gpu` suite is run once on such a build.
Where `compute-sanitizer` is open, the same module is its target:
    compute-sanitizer --tool memcheck python -m paper_2111_01064_b200.sanitize_smoke
Inputs are the seeded workloads at reduced sizes, completed with the library itself (synth.py); parity is tests/.
"""
from __future__ import annotations

import sys

import numpy as np
import torch

from . import synth, workloads as wlm
from .binding import Context, LL_PREC_FP32_ACC


def _full_families(n_c: int, log):
    dev = "cuda"
    # ---- shared nodes, one mode: small-batch route (one-warp blocks), large-batch route (> 1024 walkers), mixed precision
    wl = wlm.make_workload(0, n_w=1100, t_obs=2.0 ** 14, n_knots=40, n_c=n_c)
    ctx = synth.make_context(wl)
    b = synth.setup(ctx, wl)
    ctx.full_batch_standin(wl.f_nodes, b["params"][:70])
    ctx.full_batch_standin(wl.f_nodes, b["params"])
    ctx.standin_split_tc(True)
    ctx.full_batch_standin(wl.f_nodes, b["params"][:70])
    ctx.standin_split_tc(False)
    amp, ph, band = ctx.standin_nodes(wl.f_nodes, b["params"][:70], with_band=True)
    tf = b["params"][:70, 5:5 + 2 * n_c].reshape(70, 1, n_c, 2).contiguous()
    ts = torch.linspace(-300.0, 300.0, 70, dtype=torch.float64, device=dev)
    ctx.full_batch(wl.f_nodes, amp, ph, tf, band, t_shift=ts)
    tfn = synth.smooth_tf_nodes(b["params"][:70], wl.f_nodes, n_m=1, n_c=n_c)
    ctx.full_batch_tf(wl.f_nodes, amp, ph, tfn, band, t_shift=ts)
    xw = torch.as_tensor(np.ascontiguousarray(wl.f_nodes), device=dev).repeat(70, 1).contiguous()
    ctx.full_batch_pw(xw, amp, ph, tf, band, t_shift=ts)
    ctx.tlm_nodes(wl.f_nodes, ph, 100.0)
    ctx.full_template_standin(wl.f_nodes, wl.params[3])
    log.append(f"n_c={n_c}: full-grid single mode (small and large route), t_shift, tf, per-walker nodes: "
               f"{ctx.kernel_launches()} launches")
    if n_c == 2:
        cm = synth.make_context(wl, precision=LL_PREC_FP32_ACC)
        g = wl.grid
        cm.set_data(g.n_f, g.k_min, g.df, b["d"], b["W"])
        cm.full_batch_standin(wl.f_nodes, b["params"])
        log.append(f"FP32-accumulate variant: {cm.kernel_launches()} launches")
        assert cm.debug_check() == 0, cm.last_error()
        cm.destroy()
    assert ctx.debug_check() == 0, ctx.last_error()
    ctx.destroy()
    # ---- three modes through the generic kernels
    wl = wlm.make_workload(3, n_w=70, t_obs=2.0 ** 14, n_knots=12, n_c=n_c)
    wl.path, wl.n_m = "full", 3
    wl.modes_l, wl.modes_m, wl.c_lm = wl.modes_l[:3], wl.modes_m[:3], wl.c_lm[:3]
    P = 5 + 2 * n_c * 3
    wl.params, wl.inj = np.ascontiguousarray(wl.params[:, :P]), wl.inj[:P].copy()
    wl.f_nodes = wlm.geomspace_exact(wlm.F_LO, wlm.F_HI, 40)
    ctx = synth.make_context(wl)
    b = synth.setup(ctx, wl)
    ctx.full_batch_standin(wl.f_nodes, b["params"])
    amp, ph, band = ctx.standin_nodes(wl.f_nodes, b["params"], with_band=True)
    tfn = synth.smooth_tf_nodes(b["params"], wl.f_nodes, n_m=3, n_c=n_c)
    ctx.full_batch_tf(wl.f_nodes, amp, ph, tfn, band)
    tf = b["params"][:, 5:].reshape(70, 3, n_c, 2).contiguous()
    xw = torch.as_tensor(np.ascontiguousarray(wl.f_nodes), device=dev).repeat(70, 1).contiguous()
    ctx.full_batch_pw(xw, amp, ph, tf, band)
    if n_c == 2:  # more than 1024 walkers, three modes, the BASELINE layout: k_full_fused_hm (every mode by its own recurrence)
        big = b["params"].repeat(16, 1)[:1100].contiguous()
        ctx.full_batch_standin(wl.f_nodes, big)
    log.append(f"n_c={n_c}: full-grid three modes (generic, recurrence, tf, per-walker nodes): {ctx.kernel_launches()} launches")
    assert ctx.debug_check() == 0, ctx.last_error()
    ctx.destroy()


def _het_families(n_c: int, log):
    for index, n_w in ((1, 200), (3, 100)):
        wl = wlm.make_workload(index, n_w=n_w, t_obs=2.0 ** 15, n_knots=24, n_c=n_c)
        ctx = synth.make_context(wl)
        b = synth.setup(ctx, wl)
        p = b["params"]
        out = ctx.het_batch_standin(p)
        ctx.het_audit_standin(p[:16])
        e = torch.as_tensor(wl.f_edges, device="cuda")
        amp_e = torch.ones((n_w, wl.n_m, len(wl.f_edges)), dtype=torch.float64, device="cuda")
        ph_e = (e * 1000.0).expand(n_w, wl.n_m, -1).contiguous()
        tf = p[:, 5:].reshape(n_w, wl.n_m, n_c, 2).contiguous()
        ctx.het_batch(amp_e, ph_e, tf, t_shift=torch.zeros(n_w, dtype=torch.float64, device="cuda"))
        if index == 1:
            ctx.het_refresh_standin(p, out[0], len(wl.f_edges))
            # sampler: the multi-launch step, then the loop as one cooperative launch and as 8 launches per iteration
            n_t, n_wk = 4, 48
            x = p[: n_t * n_wk].reshape(n_t, n_wk, -1).clone()
            first = ctx.het_batch_standin(x.reshape(n_t * n_wk, -1).contiguous())
            logL, d_h, h_h = (v.reshape(n_t, n_wk).clone() for v in first)
            P = x.shape[-1]
            lo = torch.full((P,), -float("inf"), dtype=torch.float64, device="cuda")
            hi = torch.full((P,), float("inf"), dtype=torch.float64, device="cuda")
            betas = torch.tensor([1.0, 0.5, 0.2, 0.0], dtype=torch.float64, device="cuda")
            u = torch.rand((3, n_t, n_wk // 2), dtype=torch.float64, device="cuda")
            acc = torch.zeros((n_t, n_wk // 2), dtype=torch.int32, device="cuda")
            ctx.pt_stretch_half(0, x, logL, d_h, h_h, betas, lo, hi, 5, u[0], u[1], u[2], accepted=acc)
            ctx.pt_swap(x, logL, d_h, h_h, betas, torch.rand((n_t - 1, n_wk), dtype=torch.float64, device="cuda"))
            ctx.pt_stats(logL[0], d_h[0], h_h[0])
            n_acc = torch.zeros(n_t, dtype=torch.int64, device="cuda")
            ctx.pt_run(x, logL, d_h, h_h, betas, lo, hi, 5, 7, 0, 3, n_accepted=n_acc)
            ctx.pt_fused(False)
            ctx.pt_run(x, logL, d_h, h_h, betas, lo, hi, 5, 7, 3, 2, n_accepted=n_acc)
            ctx.pt_fused(True)
        log.append(f"n_c={n_c}: heterodyne config-{index} recipe ({wl.n_m} modes): {ctx.kernel_launches()} launches")
        assert ctx.debug_check() == 0, ctx.last_error()
        ctx.destroy()


def main() -> int:
    assert torch.cuda.is_available(), "needs a CUDA device (there is no CPU fallback)"
    log = []
    for n_c in (2, 3):
        _full_families(n_c, log)
        _het_families(n_c, log)
    # the sampler loop on the full-grid likelihood (small-batch route inside)
    wl = wlm.make_workload(0, n_w=64, t_obs=2.0 ** 14, n_knots=40)
    ctx = synth.make_context(wl)
    b = synth.setup(ctx, wl)
    n_t, n_wk = 2, 32
    x = b["params"].reshape(n_t, n_wk, -1).clone()
    first = ctx.full_batch_standin(wl.f_nodes, b["params"])
    logL = first[0].reshape(n_t, n_wk).clone()
    P = x.shape[-1]
    lo = torch.full((P,), -float("inf"), dtype=torch.float64, device="cuda")
    hi = torch.full((P,), float("inf"), dtype=torch.float64, device="cuda")
    betas = torch.tensor([1.0, 0.1], dtype=torch.float64, device="cuda")
    ctx.pt_run(x, logL, None, None, betas, lo, hi, 5, 11, 0, 2, f_nodes=wl.f_nodes)
    log.append(f"sampler loop on the full-grid likelihood: {ctx.kernel_launches()} launches")
    assert ctx.debug_check() == 0, ctx.last_error()
    ctx.destroy()
    torch.cuda.synchronize()
    for line in log:
        print(line)
    print("sanitize_smoke: done")
    return 0


if __name__ == "__main__":
    sys.exit(main())
