#!/usr/bin/env python
"""bench.py — log-likelihood evaluations/s of the B200-native library on BASELINE.json's workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload 2] [--quick]

A step is one pass of the whole full-grid hot path (F1-F4: parameters -> node amp/phase -> spline -> fused
evaluate/response/inner products -> log L) over BASELINE.json config 2 (16384 walkers x 1 574 725 bins, 1024
nodes, FP64), the configuration north_star sets its roofline target on.  The same JSON line carries the
heterodyned configs (1, 3, 4) and config 0 under "per_config", the ALU roofline of the fused kernel, the
end-to-end number through the C ABI with host buffers, and the CPU oracle timed on this box.

N > 1 (torchrun): walkers are independent, so every rank runs its own seeded config-2 batch
(weak scaling), no data-path collective; the time is the max over ranks, the value the sum of units / that time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2111_01064_b200 import workloads as wlm  # noqa: E402

METRIC = "log-likelihood evals/sec"
UNIT = "evals/s"
# algorithmic FP64 issue slots per active (walker, bin, mode) of the full-grid path.  Direct formulation (DESIGN.md §6:
# t 1, two cubics 6, reduce 3, sincos 18, A e^{-i Psi} 2, two complex MACs 8, W A^2 2 => 40; SURVEY.md §8(d) uses 39).
# The single-mode FP64 kernel advances e^{-i Psi} and A by recurrence (three complex rotations and three additions per
# bin, re-synchronised from the cubics every 32 bins), and SURVEY §8(d) asks that such a build quote ITS count:
# 12 + 3 + 2 + 8 + 2 = 27 per bin plus (2 cubics 6 + differences 16 + 3 sincos 54 + 3 normalisations 15 + 1)/32 = 2.9 => 30
SLOTS_FULL_DIRECT = 39.0
SLOTS_FULL = 30.0
# per-walker node grids: the recurrence route with T^c applied per bin (it accumulates <d|h>, <h|h> directly):
# 12 + 3 + 2 + T^c h 8 + Re g h 4 + W |h|^2 5 = 34 per bin + (6 + 16 + 4 sincos 72 + 20 + 1)/32 = 3.6 => 38
SLOTS_FULL_PW = 38.0
# single mode: the kernel regroups Eq. 14/17 by edge, whose own count is 48 slots per (walker, bin): phase 2,
# reduce 3, sincos 18, taper and amplitude 4, z conj(Q) 8, |z|^2 P 3, z_b conj(z_{b+1}) X 10; the bin-by-bin form needs 73
SLOTS_HET = {1: 48.0, 6: 252.0}
SLOTS_HET_DIRECT_FORM = {1: 73.0}
# FP32-accumulate variant: bound by instruction issue (one warp instruction per scheduler per
# clock = 4 x 32 lane-instructions/clk/SM).  Algorithmic instructions per active pair: 13 FP64 (t, two cubics,
# reduce 3, scale 1, W A^2 2) + 3 conversions + 20 binary32 (sincos 10, A e^{-i Psi} 2, MACs 8) + 6 quadrant
# + 2 shared loads + 1 loop = 45
INSTR_FULL_FP32ACC = 45.0
# frequency-dependent transfer function (Eq. 8-9), direct formulation: t 1, six cubics 18, reduce 3, sincos 18,
# A e^{-i Psi} 2, T^c h 8, Re g h 4, W |h|^2 5 = 59.  The kernel advances A and e^{-i Psi} by the recurrence and keeps
# Horner for the four T cubics: t 1 + 12 + rotations 12 + amplitude 3 + 2 + 8 + 4 + 5 = 47 per bin + re-sync 3 => 50
SLOTS_FULL_TF = 50.0
ISSUE_LANES_PER_CLK_PER_SM = 128.0
# DRAM traffic per launch of the dominant kernel, from the committed `ncu --set full` captures (profiles/)
NCU_TRAFFIC_BYTES = {("k_full_fused", 2): 806.3e6 + 39.9e6, ("k_full_fused_mixed", 2): 786.4e6 + 37.0e6}
DFMA_PER_CLK_PER_SM = 64.0


# ------------------------------------------------------------------------------------------------ helpers
def rank_workload(index: int, rank: int, n_w=None, **kw):
    """rank r draws its own batch: seed = SEED_BASE + index + 1000 r (weak scaling, walkers independent)."""
    return wlm.make_workload(index, n_w=n_w, seed_offset=rank, **kw)


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def allreduce_max(x: float) -> float:
    import torch
    dist = _dist()
    if dist is None:
        return float(x)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def allreduce_sum(x: float) -> float:
    import torch
    dist = _dist()
    if dist is None:
        return float(x)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([x], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def barrier():
    dist = _dist()
    if dist is not None:
        dist.barrier()


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region (pynvml; nvidia-smi as a fallback)."""

    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4, "hw_power_brake": 0x80}

    def __init__(self, index: int, period: float = 0.02):
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._t = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)) if hasattr(
                    nv, "nvmlDeviceGetCurrentClocksEventReasons") else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in {**self.BAD, **self.NOTE}.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._t = threading.Thread(target=self._loop, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._t is not None:
            self._t.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)), "measured"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


# ------------------------------------------------------------------------------------------------ GPU arm
def time_steps(torch, fn, steps: int, warmup: int):
    """W untimed steps, then K steps between two events on the current stream; returns total ms."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1)


def bench_config(torch, index: int, steps: int, warmup: int, rank: int = 0, profile: bool = False, precision: int = 0):
    """device-resident timing of one config through the stand-in entry point (parameters -> log L).
    precision = 1: the FP32-accumulate variant of the full-grid path on the SAME data (the data stream is built
    by an FP64 context first, so the two variants can be compared output by output)."""
    from paper_2111_01064_b200 import synth
    wl = rank_workload(index, rank)
    ctx = synth.make_context(wl)
    bufs = synth.setup(ctx, wl)
    if precision:
        ctx.destroy()
        ctx = synth.make_context(wl, precision=precision)
        g = wl.grid
        ctx.set_data(g.n_f, g.k_min, g.df, bufs["d"], bufs["W"])
    params = bufs["params"]
    n_w = wl.n_w
    out = tuple(torch.empty(n_w, dtype=torch.float64, device=params.device) for _ in range(3))
    if wl.path == "full":
        fn = lambda: ctx.full_batch_standin(wl.f_nodes, params, out=out)
    else:
        fn = lambda: ctx.het_batch_standin(params, out=out)
    fn()                                    # first call: workspace allocation
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    l0 = ctx.kernel_launches()
    if profile:
        ctx.profile_enable(True)
    ms = time_steps(torch, fn, steps, 0)
    res = {"wl": wl, "ctx": ctx, "bufs": bufs, "fn": fn, "out": out, "ms_total": ms, "ms_per_step": ms / steps,
           "launches": ctx.kernel_launches() - l0}
    if profile:
        kms, kn = ctx.profile_read()
        ctx.profile_enable(False)
        res["kernel_ms"] = kms / max(kn, 1)
        res["kernel_n"] = kn
    return res


def bench_sampler_iteration(torch, ctx, wl, params, n_t: int = 10, n_w: int = 400, iters: int = 50, f_nodes=None):
    """one sampler iteration — two half updates (propose, likelihood, accept), a temperature-swap
    sweep and the stopping statistics — timed eagerly and as a CUDA-graph replay (the iteration never returns to the
    host).  Default: Module-2 size (10 temperatures x 400 walkers) on the heterodyned likelihood;
    with f_nodes: the full-grid likelihood (Module 1: 4 temperatures x 80 walkers)."""
    P = params.shape[1]
    x = params[: n_t * n_w].reshape(n_t, n_w, P).clone()
    x[:, :, 5:] = params[0, 5:]                      # transfer factors frozen: 5 sampled coordinates
    flat = x.reshape(-1, P)
    c = flat[:, :5].mean(dim=0)
    w = 3.0 * (flat[:, :5].max(dim=0).values - flat[:, :5].min(dim=0).values)
    lo = torch.full((P,), -float("inf"), dtype=torch.float64, device=x.device)
    hi = torch.full((P,), float("inf"), dtype=torch.float64, device=x.device)
    lo[:5], hi[:5] = c - w, c + w
    betas = torch.tensor([0.5 ** t for t in range(n_t - 1)] + [0.0], dtype=torch.float64, device=x.device)
    first = ctx.het_batch_standin(flat.contiguous()) if f_nodes is None else ctx.full_batch_standin(f_nodes, flat.contiguous())
    logL, d_h, h_h = (v.reshape(n_t, n_w).clone() for v in first)
    out3 = torch.empty(3, dtype=torch.float64, device=x.device)
    acc = torch.zeros((n_t, n_w // 2), dtype=torch.int32, device=x.device)
    n_acc = torch.zeros((), dtype=torch.int64, device=x.device)

    def iteration():
        for half in (0, 1):
            u = torch.rand((3, n_t, n_w // 2), dtype=torch.float64, device=x.device)
            ctx.pt_stretch_half(half, x, logL, d_h, h_h, betas, lo, hi, 5, u[0], u[1], u[2], accepted=acc, f_nodes=f_nodes)
            n_acc.add_(acc.sum())
        ctx.pt_swap(x, logL, d_h, h_h, betas, torch.rand((n_t - 1, n_w), dtype=torch.float64, device=x.device))
        ctx.pt_stats(logL[0], d_h[0], h_h[0], out3=out3)

    for _ in range(5):
        iteration()
    ms_eager = time_steps(torch, iteration, iters, 0) / iters
    res = {"n_temps": n_t, "n_walkers": n_w,
           "likelihood": ("heterodyned, %d bins" % (len(wl.f_edges) - 1)) if f_nodes is None else
                         ("full grid, %d bins, %d nodes" % (wl.grid.n_f, len(f_nodes))),
           "ms_per_iteration_eager": ms_eager, "evals_per_s_eager": n_t * n_w / (ms_eager * 1e-3)}
    try:
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            iteration()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=s):
                iteration()
        torch.cuda.current_stream().wait_stream(s)
        n_acc.zero_()
        ms_graph = time_steps(torch, graph.replay, iters, 3) / iters
        res.update({"ms_per_iteration_graph": ms_graph, "evals_per_s_graph": n_t * n_w / (ms_graph * 1e-3),
                    "acceptance_fraction": float(n_acc) / ((iters + 3) * n_t * n_w),
                    "max_logL_cold_chain": float(out3[0]), "extracted_snr_cold_chain": float(out3[2])})
    except Exception as e:  # capture is a convenience of the harness, not part of the library
        res["graph_error"] = repr(e)[:200]
    # ---- the library's own loop: ll_pt_run_* (counter-based uniforms, nothing returns to the host), in blocks of 150
    # iterations with the stopping statistics read back after each block, as the paper's modules do
    from paper_2111_01064_b200 import binding
    n_acc64 = torch.zeros(n_t, dtype=torch.int64, device=x.device)
    stop = binding.StopState(n_checks=30, tol=1.0)
    blocks, per_block = (4, 150) if f_nodes is None else (2, 20)
    ctx.pt_run(x, logL, d_h, h_h, betas, lo, hi, 5, 2111, 0, 5, f_nodes=f_nodes)          # warm-up
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for b in range(blocks):
        ctx.pt_run(x, logL, d_h, h_h, betas, lo, hi, 5, 2111, 5 + b * per_block, per_block, n_accepted=n_acc64, f_nodes=f_nodes)
        st3 = ctx.pt_stats(logL[0], d_h[0], h_h[0], out3=out3).cpu()                        # synchronises
        stopped = binding.stop_converged(stop, float(st3[0])) or binding.stop_snr(float(st3[2]), float("inf"))
    ms_run = (time.perf_counter() - t0) * 1e3 / (blocks * per_block)
    res.update({"ms_per_iteration_run": ms_run, "evals_per_s_run": n_t * n_w / (ms_run * 1e-3),
                "run": "ll_pt_run_%s, %d blocks of %d iterations, stopping statistics read back after each (host wall time)"
                       % ("het" if f_nodes is None else "full", blocks, per_block),
                "acceptance_fraction_run": float(n_acc64.sum()) / (blocks * per_block * n_t * n_w), "stopped": bool(stopped)})
    return res


def bench_full_hm(torch, steps: int = 5, n_w: int = 2048):
    """The paper's higher-mode analysis ran the brute-force likelihood, not the heterodyned one: config 3's
    six modes through the FULL-GRID path on config 2's one-year grid and 1024 nodes, prior-draw walkers with unit-modulus
    transfer factors per mode, data = noise of the config-2 recipe (timing only; parity of this path is in the tests)."""
    from paper_2111_01064_b200 import binding
    wl6, wl2 = wlm.make_workload(3, n_w=8), wlm.make_workload(2, n_w=n_w)
    rng = np.random.default_rng(wlm.SEED_BASE + 232)
    params = np.empty((n_w, 5 + 4 * wl6.n_m))
    params[:, :5] = wl2.params[:, :5]
    ang = rng.uniform(0, 2 * np.pi, (n_w, 2 * wl6.n_m))
    params[:, 5::2], params[:, 6::2] = np.cos(ang), np.sin(ang)
    ctx = binding.Context(n_modes=wl6.n_m)
    ctx.standin_config(wl6.modes_l, wl6.modes_m, wl6.c_lm, wl6.kappa)
    g = wl2.grid
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")
    ctx.set_data(g.n_f, g.k_min, g.df, dev(wl2.noise), dev(wl2.W))
    p = dev(params)
    out = tuple(torch.empty(n_w, dtype=torch.float64, device="cuda") for _ in range(3))
    fn = lambda: ctx.full_batch_standin(wl2.f_nodes, p, out=out)
    fn()
    ctx.profile_enable(True)
    ms = time_steps(torch, fn, steps, 2) / steps
    kms, kn = ctx.profile_read()
    pairs = ctx.last_full_stats()[0]
    ctx.destroy()
    return {"evals_per_s": n_w / (ms * 1e-3), "ms_per_batch": ms, "n_walkers": n_w, "n_modes": int(wl6.n_m),
            "kernel": "k_full_fused<0>", "kernel_ms": kms / max(kn, 1), "active_pair_modes": pairs,
            "algorithmic_slots_per_pair_mode": SLOTS_FULL_DIRECT}


def e2e_config(torch, res, steps: int, warmup: int):
    """same metric through the C ABI with HOST buffers: pinned params in, pinned results out, every step."""
    wl, ctx = res["wl"], res["ctx"]
    ph = torch.as_tensor(np.ascontiguousarray(wl.params)).pin_memory()
    outs = tuple(torch.empty(wl.n_w, dtype=torch.float64).pin_memory() for _ in range(3))
    if wl.path == "full":
        fn = lambda: ctx.full_batch_standin_host(wl.f_nodes, ph, outs)
    else:
        fn = lambda: ctx.het_batch_standin_host(ph, outs)
    ms = time_steps(torch, fn, steps, warmup)
    dev_logL = res["out"][0].cpu()
    assert torch.equal(dev_logL, outs[0]), "host-buffer path and device-resident path disagree"
    return ms / steps, ph.numel() * 8, 3 * wl.n_w * 8


def cpu_baseline(index: int, n_sample: int, budget_note: str = ""):
    """the oracle, as it stands, on this box's cores, on the first n_sample walkers of the same workload"""
    import oracle as orc
    wl = rank_workload(index, 0)
    g = wl.grid
    t_setup = time.perf_counter()
    if wl.path == "full":
        run = lambda p, d, t=False: orc.full_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, p, wl.f_nodes, g.k_min, g.df,
                                                           g.n_f, d, wl.W, want_template=t)
        wl.finish_distance(run(wl.inj[None], None)["h_h"][0])
        d = wl.make_data(run(wl.inj[None], None, True)["h"])
        work = lambda: run(wl.params[:n_sample], d)
    else:
        f = g.freqs()
        direct = lambda p, ff: orc.standin_direct(p, wl.modes_m, wl.c_lm, wl.kappa, ff, float(f[0]), float(f[-1]))
        h1 = direct(wl.inj, f)
        wl.finish_distance(orc.inner(h1, h1, wl.W).real)
        h0 = direct(wl.inj, f)
        d = wl.make_data(h0)
        h0e = direct(wl.inj, wl.f_edges)
        summ = orc.het_prepare(g.k_min, g.df, d, wl.W, h0, wl.f_edges)
        work = lambda: orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params[:n_sample], wl.f_edges, h0e, summ)
    t_setup = time.perf_counter() - t_setup
    t0 = time.perf_counter()
    work()
    dt = time.perf_counter() - t0
    return {"value": n_sample / dt, "unit": UNIT, "cores": orc.n_threads(), "kind": "oracle",
            "sample": f"{wl.name}: first {n_sample} of {wl.n_w} walkers, whole grid, {dt:.1f} s wall{budget_note}",
            "seconds": dt, "work": work, "n_sample": n_sample}


def run_reference(args):
    """--impl reference: the oracle is the reference arm for this tier (no reference implementation exists)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle as orc
    orc.build()
    cores = orc.n_threads()
    n_sample = max(cores, 1)
    cb = cpu_baseline(args.workload, n_sample)
    work = cb.pop("work")
    for _ in range(max(args.warmup - 1, 0)):
        work()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        work()
    dt = time.perf_counter() - t0
    wl = rank_workload(args.workload, 0)
    val = n_sample * args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 (x87 long double accumulators)", "data": "synthetic",
            "config": workload_config(wl, extra={"step": f"{n_sample} walkers of the batch per step (bounded sample)"}),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{wl.name}: first {n_sample} walkers per step, whole grid"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def workload_config(wl, extra=None):
    g = wl.grid
    c = {"workload": wl.name, "path": wl.path, "n_walkers": wl.n_w, "n_modes": wl.n_m, "n_channels": wl.n_c,
         "n_f": g.n_f, "t_obs_s": g.t_obs,
         "inputs": "seeded synthetic (DESIGN.md §4), stand-in for LDC-1A",
         "l2": "working set (spline coefficients 1.07 GB + node values 0.27 GB per step) exceeds the 126 MB L2; "
               "no flush needed"}
    if wl.path == "full":
        c["n_nodes"] = int(len(wl.f_nodes))
    else:
        c["n_bins"] = int(len(wl.f_edges) - 1)
        c["l2"] = "params and outputs only; summary tables live in shared memory (nothing to flush)"
    if extra:
        c.update(extra)
    return c


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", type=int, default=2, help="BASELINE.json config index of the headline step")
    ap.add_argument("--quick", action="store_true", help="skip per_config, e2e and cpu_baseline (profiling runs)")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32acc"],
                    help="fp32acc: time the FP32-accumulate variant of the full-grid path as the headline step")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    if args.impl == "reference":
        return run_reference(args)

    import torch
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    from paper_2111_01064_b200 import build as _b
    if rank == 0 or not os.path.exists(_b.SO):
        _b.build()
    barrier()

    peaks, peak_src = measured_peaks()
    with ClockSampler(local) as clk:
        res = bench_config(torch, args.workload, args.steps, args.warmup, rank=rank, profile=True,
                           precision=1 if args.precision == "fp32acc" else 0)
    wl, ctx = res["wl"], res["ctx"]
    headline_logL = res["out"][0].clone()
    t_ms = allreduce_max(res["ms_total"])
    units = allreduce_sum(float(wl.n_w) * args.steps)
    value = units / (t_ms * 1e-3)
    clocks = clk.summary()

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if args.precision == "fp64" else "f64 phase/amplitude/<h|h> + f32 trig/products (reading R15)",
            "data": "synthetic", "config": workload_config(wl), "clocks": clocks,
            "gpu_launches": int(res["launches"]), "impl": "b200"}

    if rank == 0:
        # ---- roofline of the dominant kernel (fused full-grid F3, or the het batch kernel)
        sm_max = float(clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz", 1965.0))
        n_sm = torch.cuda.get_device_properties(local).multi_processor_count
        peak_slots = n_sm * DFMA_PER_CLK_PER_SM * sm_max * 1e6
        if wl.path == "full":
            pairs, n_blocks = ctx.last_full_stats()
            slots = pairs * SLOTS_FULL
            kname = "k_full_fused" if args.precision == "fp64" else "k_full_fused_mixed"
        else:
            pairs = float(wl.n_w) * (len(wl.f_edges) - 1)
            slots = pairs * SLOTS_HET.get(wl.n_m, 73.0 + 36.0 * (wl.n_m - 1))
            kname = "k_het_standin"
        k_ms = res["kernel_ms"]
        dfma_rate, dfma_ms = ctx.peak_fma(0, 4000)
        ffma_rate, _ = ctx.peak_fma(1, 8000)
        traffic = NCU_TRAFFIC_BYTES.get((kname, args.workload))
        if kname == "k_full_fused_mixed":
            peak_issue = n_sm * ISSUE_LANES_PER_CLK_PER_SM * sm_max * 1e6
            achieved = pairs * INSTR_FULL_FP32ACC / (k_ms * 1e-3)
            line["roofline"] = {
                "bound": "alu", "kernel": kname, "achieved": achieved / 1e12, "peak": peak_issue / 1e12,
                "unit": "T lane-instructions/s (instruction issue: 1 warp instruction/scheduler/clk)",
                "frac": achieved / peak_issue, "traffic": traffic, "kernel_ms": k_ms,
                "kernel_share_of_step": k_ms / (res["ms_per_step"]),
                "algorithmic_instructions_per_pair": INSTR_FULL_FP32ACC, "active_pairs": pairs,
                "peak_source": f"{n_sm} SMs x 4 schedulers x 32 lanes x {sm_max:.0f} MHz (DESIGN.md §6)",
                "fp64_slots_per_pair": 13.0, "fp64_pipe_frac": pairs * 13.0 / (k_ms * 1e-3) / peak_slots,
                "measured_dfma_per_s": dfma_rate, "measured_ffma_per_s": ffma_rate,
                "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peak_src}
        else:
            achieved = slots / (k_ms * 1e-3)
            line["roofline"] = {
                "bound": "alu", "kernel": kname, "achieved": achieved / 1e12, "peak": peak_slots / 1e12,
                "unit": "T FP64 issue slots/s (1 DFMA|DMUL|DADD = 1 slot)", "frac": achieved / peak_slots,
                "traffic": traffic, "kernel_ms": k_ms, "kernel_share_of_step": k_ms / (res["ms_per_step"]),
                "algorithmic_slots_per_pair": SLOTS_FULL if wl.path == "full" else slots / pairs, "active_pairs": pairs,
                "peak_source": f"{n_sm} SMs x {int(DFMA_PER_CLK_PER_SM)} DFMA/clk x {sm_max:.0f} MHz (DESIGN.md §6)",
                "measured_dfma_per_s": dfma_rate, "measured_ffma_per_s": ffma_rate,
                "frac_of_measured_dfma": achieved / dfma_rate,
                "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peak_src}
            if wl.path == "full":
                line["roofline"]["formulation"] = ("rotation recurrence, re-synchronised every 32 bins (DESIGN.md §5); the direct "
                                                   "formulation needs %g slots per pair" % SLOTS_FULL_DIRECT)
                line["roofline"]["frac_in_direct_form_slots"] = pairs * SLOTS_FULL_DIRECT / (k_ms * 1e-3) / peak_slots
            if wl.path != "full" and wl.n_m in SLOTS_HET_DIRECT_FORM:
                line["roofline"]["formulation"] = "regrouped by edge (DESIGN.md §5); the bin-by-bin form of Eq. 14/17 needs %g" \
                                                  % SLOTS_HET_DIRECT_FORM[wl.n_m]

    if not args.quick:
        # ---- end to end through the C ABI with host buffers
        ms_e2e, bi, bo = e2e_config(torch, res, max(args.steps // 2, 3), 3)
        t_e2e = allreduce_max(ms_e2e)
        line["e2e"] = {"value": world * wl.n_w / (t_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": bi,
                       "d2h_bytes_per_step": bo, "ms_per_step": t_e2e}
    res["ctx"].destroy()
    del res
    torch.cuda.empty_cache()

    if rank == 0 and not args.quick and world == 1:
        # ---- every BASELINE.json config, device-resident, stand-in entry points
        per = {}
        for idx in (0, 1, 2, 3, 4):
            if idx == args.workload:
                per[f"cfg{idx}"] = {"evals_per_s": value, "ms_per_batch": t_ms / args.steps, "n_walkers": wl.n_w}
                continue
            st = 50 if idx != 2 else args.steps
            r = bench_config(torch, idx, st, 5)
            per[f"cfg{idx}"] = {"evals_per_s": r["wl"].n_w / (r["ms_per_step"] * 1e-3), "ms_per_batch": r["ms_per_step"],
                                "n_walkers": r["wl"].n_w}
            if idx in (0, 1):
                # ---- launch-bound configs: the same call replayed as a CUDA graph
                try:
                    sg = torch.cuda.Stream()
                    sg.wait_stream(torch.cuda.current_stream())
                    with torch.cuda.stream(sg):
                        r["fn"]()
                        gr = torch.cuda.CUDAGraph()
                        with torch.cuda.graph(gr, stream=sg):
                            r["fn"]()
                    torch.cuda.current_stream().wait_stream(sg)
                    ms_g = time_steps(torch, gr.replay, 200, 5) / 200
                    per[f"cfg{idx}"].update({"ms_per_batch_graph": ms_g, "evals_per_s_graph": r["wl"].n_w / (ms_g * 1e-3)})
                    del gr
                except Exception as e:
                    per[f"cfg{idx}"]["graph_error"] = repr(e)[:200]
            if idx == 1:
                # ---- the reference update inside the loop (every 5000 iterations)
                # and the brute-force audit of the heterodyned values, config-1 size
                c1, p1, n_e = r["ctx"], r["bufs"]["params"], len(r["wl"].f_edges)
                t0 = time.perf_counter()
                for _ in range(5):
                    c1.het_refresh_standin(p1, r["out"][0], n_e)          # synchronises the stream itself
                ms_ref = (time.perf_counter() - t0) / 5 * 1e3
                het = [x.clone() for x in c1.het_batch_standin(p1)]
                o1 = tuple(torch.empty_like(het[0]) for _ in range(3))
                ms_a = time_steps(torch, lambda: c1.het_audit_standin(p1, out=o1), 5, 2) / 5
                per["cfg1_refresh"] = {"ms_per_update": ms_ref, "n_edges": n_e, "n_f": r["wl"].grid.n_f,
                                       "entry": "ll_het_refresh_standin (argmax, h0 on the grid and at the edges, H0; host wall time, the call synchronises)"}
                per["cfg1_audit"] = {"evals_per_s": r["wl"].n_w / (ms_a * 1e-3), "ms_per_batch": ms_a, "n_walkers": r["wl"].n_w,
                                     "max_abs_het_minus_dense_logL": float((het[0] - o1[0]).abs().max()),
                                     "entry": "ll_het_audit_standin (direct template at every dense bin of the band)"}
                per["module2_iteration"] = bench_sampler_iteration(torch, c1, r["wl"], p1)
            r["ctx"].destroy()
            del r
            torch.cuda.empty_cache()
        if args.workload == 2 and args.precision == "fp64":
            # ---- config 2's FP32-accumulate variant on the same data: throughput and its distance from FP64
            r = bench_config(torch, 2, args.steps, 5, profile=True, precision=1)
            dl = (r["out"][0] - headline_logL).abs()
            per["cfg2_fp32acc"] = {"evals_per_s": r["wl"].n_w / (r["ms_per_step"] * 1e-3), "ms_per_batch": r["ms_per_step"],
                                   "n_walkers": r["wl"].n_w, "kernel": "k_full_fused_mixed", "kernel_ms": r["kernel_ms"],
                                   "max_abs_dlogL_vs_fp64": float(dl.max()), "rms_dlogL_vs_fp64": float(dl.pow(2).mean().sqrt())}
            r["ctx"].destroy()
            del r
            torch.cuda.empty_cache()
        if args.workload == 2 and args.precision == "fp64":
            # ---- frequency-dependent transfer function (six splines per mode) at config-2
            # size through the array entry point; node arrays from ll_standin_nodes, a smooth T(f) at the nodes
            from paper_2111_01064_b200 import synth
            wl2 = rank_workload(2, 0)
            c2 = synth.make_context(wl2)
            b2 = synth.setup(c2, wl2)
            amp, ph, bnd = c2.standin_nodes(wl2.f_nodes, b2["params"], with_band=True)
            tfn = synth.smooth_tf_nodes(b2["params"], wl2.f_nodes)
            o2 = tuple(torch.empty(wl2.n_w, dtype=torch.float64, device=amp.device) for _ in range(3))
            fn2 = lambda: c2.full_batch_tf(wl2.f_nodes, amp, ph, tfn, band=bnd, out=o2)
            fn2()
            c2.profile_enable(True)
            ms2 = time_steps(torch, fn2, max(args.steps // 2, 3), 3)
            kms, kn = c2.profile_read()
            c2.profile_enable(False)
            nst = max(args.steps // 2, 3)
            pairs2 = c2.last_full_stats()[0]
            per["cfg2_tf"] = {"evals_per_s": wl2.n_w / (ms2 / nst * 1e-3), "ms_per_batch": ms2 / nst, "n_walkers": wl2.n_w,
                              "kernel": "k_full_fused_tf", "kernel_ms": kms / max(kn, 1), "active_pairs": pairs2,
                              "algorithmic_slots_per_pair": SLOTS_FULL_TF,
                              "frac": pairs2 * SLOTS_FULL_TF / (kms / max(kn, 1) * 1e-3) / peak_slots,
                              "entry": "ll_full_batch_tf (amp, phase, T at 1024 nodes as device arrays; the walkers' own bands)"}
            # ---- per-walker node grids at config-2 size.  Every walker gets its own copy of the
            # 1024 nodes (so the numbers can be compared with the shared-node path output by output); what is timed is
            # the per-walker machinery: one tridiagonal factorisation per system, one bin -> interval map per lane
            tfc = b2["params"][:, 5:9].reshape(-1, 1, 2, 2).contiguous()
            xw = torch.as_tensor(np.ascontiguousarray(wl2.f_nodes), device=amp.device).repeat(wl2.n_w, 1).contiguous()
            o3 = tuple(torch.empty(wl2.n_w, dtype=torch.float64, device=amp.device) for _ in range(3))
            fn3 = lambda: c2.full_batch_pw(xw, amp, ph, tfc, band=bnd, out=o3)
            fn3()
            sh = c2.full_batch(wl2.f_nodes, amp, ph, tfc, band=bnd)
            c2.profile_enable(True)
            ms3 = time_steps(torch, fn3, nst, 2)
            kms3, kn3 = c2.profile_read()
            c2.profile_enable(False)
            per["cfg2_pw"] = {"evals_per_s": wl2.n_w / (ms3 / nst * 1e-3), "ms_per_batch": ms3 / nst, "n_walkers": wl2.n_w,
                              "kernel": "k_full_fused_pw", "kernel_ms": kms3 / max(kn3, 1),
                              "frac": pairs2 * SLOTS_FULL_PW / (kms3 / max(kn3, 1) * 1e-3) / peak_slots,
                              "algorithmic_slots_per_pair": SLOTS_FULL_PW,
                              "max_abs_dlogL_vs_shared_nodes": float((o3[0] - sh[0]).abs().max()),
                              "entry": "ll_full_batch_pw (f_nodes_w [n_w][1024] on the device; the walkers' own bands)"}
            del xw, sh, tfc
            # ---- six modes through the full-grid path (the paper's higher-mode run used the brute-force likelihood)
            hm = bench_full_hm(torch)
            hm["frac"] = hm["active_pair_modes"] * SLOTS_FULL_DIRECT / (hm["kernel_ms"] * 1e-3) / peak_slots
            per["cfg2_hm6"] = hm
            # ---- Module-1 sized sampler iteration on the full-grid likelihood of the same one-year data stream
            per["module1_iteration"] = bench_sampler_iteration(torch, c2, wl2, b2["params"], n_t=4, n_w=80, iters=20,
                                                               f_nodes=wl2.f_nodes)
            c2.destroy()
            del amp, ph, tfn, b2
            torch.cuda.empty_cache()
        line["per_config"] = per
        # ---- the oracle on this box's cores, bounded sample of the same workload
        import oracle as orc
        orc.build()
        n_sample = 4 * orc.n_threads() if wl.path == "full" else min(wl.n_w, 4096)
        cb = cpu_baseline(args.workload, n_sample)
        cb.pop("work")
        line["cpu_baseline"] = cb
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
