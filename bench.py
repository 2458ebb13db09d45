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
# Algorithmic FP64 issue slots per unit (1 DFMA | DMUL | DADD = 1 slot).
# Full grid, per active (walker, bin, mode).  Direct formulation: t 1, two cubics 6, reduce 3, sincos 18, A e^{-i Psi} 2,
# two complex MACs 8, W A^2 2 => 39.  The single-mode FP64 kernels advance e^{-i Psi} and A by recurrence, and
# SURVEY §8(d) asks that such a build quote ITS count: 12 (three rotations) + 3 (amplitude differences) + 2 (A z) +
# 4 n_c (MACs) + 2 (W A^2; 1 + n_c with per-channel weights) => 27 for two channels sharing a weight row, 33 for
# three channels with their own rows.  `frac` uses these.  The re-synchronisation every 128 bins (2 cubics 6 +
# differences 16 + 3 degree-7 sincos 57 + 3 normalisations 15 + 1 = 95 slots / 128 bins = 0.74) is the builder's tuning
# choice, not algorithmic work: `frac_with_resync` adds it and is reported beside `frac`, never instead of it.
SLOTS_FULL_DIRECT = 39.0
# several modes, large batches (k_full_fused_hm): every mode by the recurrence — 12 rotations + 3 amplitude differences + 2 A z +
# 8 T^c h = 25 per (bin, mode) — plus per bin Re(g^c h^c) 4 and W |h^c|^2 6
def slots_full_hm(n_m: int) -> float:
    return 25.0 + 10.0 / n_m
SLOTS_FULL = 27.0
SLOTS_FULL_NC3 = 33.0
SLOTS_RESYNC = 0.74
# per-walker node grids: the recurrence route with T^c applied per bin (it accumulates <d|h>, <h|h> directly):
# 12 + 3 + 2 + T^c h 8 + Re g h 4 + W |h|^2 5 = 34 per bin (+ re-sync with four sincos: 3.6)
SLOTS_FULL_PW = 34.0
# single mode: the kernel regroups Eq. 14/17 by edge, whose own count is 48 slots per (walker, bin): phase 2,
# reduce 3, sincos 18, taper and amplitude 4, z conj(Q) 8, |z|^2 P 3, z_b conj(z_{b+1}) X 10; the bin-by-bin form of
# SURVEY §8(d) needs 73.  Six modes: SURVEY's 252 (6 x 36 + 36)
SLOTS_HET = {1: 48.0, 6: 252.0}
SLOTS_HET_SURVEY_FORM = {1: 73.0, 6: 252.0}
# FP32-accumulate variant: bound by instruction issue (one warp instruction per scheduler per
# clock = 4 x 32 lane-instructions/clk/SM).  Algorithmic instructions per active pair: 13 FP64 (t, two cubics,
# reduce 3, scale 1, W A^2 2) + 3 conversions + 20 binary32 (sincos 10, A e^{-i Psi} 2, MACs 8) + 6 quadrant
# + 2 shared loads + 1 loop = 45
INSTR_FULL_FP32ACC = 45.0
# frequency-dependent transfer function (Eq. 8-9), direct formulation: t 1, six cubics 18, reduce 3, sincos 18,
# A e^{-i Psi} 2, T^c h 8, Re g h 4, W |h|^2 5 = 59.  The kernel advances A and e^{-i Psi} by the recurrence and keeps
# Horner for the four T cubics: t 1 + 12 + rotations 12 + amplitude 3 + 2 + 8 + 4 + 5 = 47 per bin
SLOTS_FULL_TF = 47.0
ISSUE_LANES_PER_CLK_PER_SM = 128.0
DFMA_PER_CLK_PER_SM = 64.0
# the parity test that covers each timed configuration at its full size (tests/, -m gpu)
COVERED_BY = {
    "cfg0": "tests/test_parity_gpu.py::test_cfg0_full_standin_parity",
    "cfg1": "tests/test_parity_gpu.py::test_cfg1_full_size",
    "cfg2": "tests/test_parity_cfg2_scale.py::test_cfg2_full_size_128_walkers",
    "cfg3": "tests/test_parity_gpu.py::test_cfg3_higher_modes_full_size_sampled",
    "cfg4": "tests/test_parity_gpu.py::test_cfg4_large_batch_full_size_sampled",
    "cfg2_fp32acc": "tests/test_parity_gpu.py::test_cfg2_full_size_sampled_mixed",
    "cfg2_tf": "tests/test_parity_cfg2_scale.py::test_cfg2_tf_full_size_sampled",
    "cfg2_pw": "tests/test_parity_cfg2_scale.py::test_cfg2_pw_full_size_sampled",
    "cfg2_hm6": "tests/test_parity_cfg2_scale.py::test_cfg2_hm6_full_size_sampled",
    "cfg2_nc3": "tests/test_parity_cfg2_scale.py::test_cfg2_three_channels_full_size_sampled",
    "cfg2_split_tc": "tests/test_parity_cfg2_scale.py::test_cfg2_split_tc_full_size_sampled",
    "module1_iteration": "tests/test_parity_cfg2_scale.py::test_module1_sized_batches_against_oracle, "
                         "tests/test_parity_gpu.py::test_pt_run_parity_full",
    "module2_iteration": "tests/test_parity_gpu.py::test_pt_run_parity_het",
}


def ncu_traffic_bytes(kernel_tag: str):
    """DRAM read + write bytes per launch of a kernel from the newest committed `ncu --set full` summary under profiles/
    whose name carries `kernel_tag` (e.g. 'full_fused_cfg2'): a measurement of THIS build's kernel, by file name, or None."""
    import glob
    import re
    cands = sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_{kernel_tag}.md")))
    if not cands:
        return None, None
    path = cands[-1]
    unit = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    tot, seen = 0.0, 0
    for line in open(path):
        m = re.match(r"\|\s*dram__bytes_(read|write)\.sum\s*\|\s*(\w+)\s*\|\s*([0-9.eE+-]+)\s*\|", line)
        if m and m.group(2) in unit:
            tot += float(m.group(3)) * unit[m.group(2)]
            seen += 1
    return (tot, os.path.relpath(path, ROOT)) if seen == 2 else (None, None)


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


def bench_config(torch, index: int, steps: int, warmup: int, rank: int = 0, profile: bool = False, precision: int = 0,
                 n_w=None, n_c=None):
    """device-resident timing of one config through the stand-in entry point (parameters -> log L).
    precision = 1: the FP32-accumulate variant of the full-grid path on the SAME data (the data stream is built
    by an FP64 context first, so the two variants can be compared output by output)."""
    from paper_2111_01064_b200 import synth
    wl = rank_workload(index, rank, n_w=n_w, **({"n_c": n_c} if n_c else {}))
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
    if f_nodes is None:
        # the same loop as 8 launches per iteration (ll_pt_fused(0)), for comparison with the one-launch form above
        ctx.pt_fused(False)
        ctx.pt_run(x, logL, d_h, h_h, betas, lo, hi, 5, 2111, 5, 5)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        ctx.pt_run(x, logL, d_h, h_h, betas, lo, hi, 5, 2111, 1000, per_block)
        torch.cuda.synchronize()
        res["ms_per_iteration_run_multi_launch"] = (time.perf_counter() - t1) * 1e3 / per_block
        ctx.pt_fused(True)
    res.update({"ms_per_iteration_run": ms_run, "evals_per_s_run": n_t * n_w / (ms_run * 1e-3),
                "run": "ll_pt_run_%s%s, %d blocks of %d iterations, stopping statistics read back after each (host wall time)"
                       % ("het" if f_nodes is None else "full", " (one cooperative launch per block of iterations)" if f_nodes is None else "",
                          blocks, per_block),
                "acceptance_fraction_run": float(n_acc64.sum()) / (blocks * per_block * n_t * n_w), "stopped": bool(stopped)})
    return res


def bench_small_batch(torch, ctx, wl, params, peak_slots, n_w: int = 160, steps: int = 20):
    """one Module-1 sized likelihood call (a half update of 4 x 80 walkers is 160 proposals): batch time
    and the fused kernel's own time and ALU-roofline fraction"""
    p = params[:n_w].contiguous()
    out = tuple(torch.empty(n_w, dtype=torch.float64, device=p.device) for _ in range(3))
    fn = lambda: ctx.full_batch_standin(wl.f_nodes, p, out=out)
    fn()
    ctx.profile_enable(True)
    ms = time_steps(torch, fn, steps, 3) / steps
    kms, kn = ctx.profile_read()
    ctx.profile_enable(False)
    pairs = ctx.last_full_stats()[0]
    k = kms / max(kn, 1)
    return {"call_%d" % n_w: {"n_walkers": n_w, "ms_per_batch": ms, "kernel_ms": k, "units": pairs, "slots_per_unit": SLOTS_FULL,
                              "frac": pairs * SLOTS_FULL / (k * 1e-3) / peak_slots}}


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
            "kernel": "k_full_fused_hm<6, 2, true>", "kernel_ms": kms / max(kn, 1), "active_pair_modes": pairs,
            "algorithmic_slots_per_pair_mode": slots_full_hm(int(wl6.n_m)),
            "formulation": "rotation recurrence per mode (25 per (bin, mode) + 10 per bin); the direct formulation of SURVEY §8(d) "
                           "needs 39 per (bin, mode) and its kernel 24.2 ms for this batch"}


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


CPU_SAMPLE_CFG2 = 128   # walkers of config 2 the oracle is timed on (>= 128)


def oracle_job(index: int, n_sample=None):
    """the oracle, as it stands, on workload `index`: returns (work(n) -> None over the first n walkers, n_total, name).
    Het configs run in full; config 2 on its first CPU_SAMPLE_CFG2 walkers over the whole grid (bounded sample)."""
    import oracle as orc
    wl = rank_workload(index, 0)
    g = wl.grid
    if wl.path == "full":
        run = lambda p, d, t=False: orc.full_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, p, wl.f_nodes, g.k_min, g.df,
                                                           g.n_f, d, wl.W, want_template=t)
        wl.finish_distance(run(wl.inj[None], None)["h_h"][0])
        d = wl.make_data(run(wl.inj[None], None, True)["h"])
        work = lambda n: run(wl.params[:n], d)
        n_total = min(wl.n_w, n_sample or (CPU_SAMPLE_CFG2 if index == 2 else wl.n_w))
    else:
        f = g.freqs()
        direct = lambda p, ff: orc.standin_direct(p, wl.modes_m, wl.c_lm, wl.kappa, ff, float(f[0]), float(f[-1]))
        h1 = direct(wl.inj, f)
        wl.finish_distance(orc.inner(h1, h1, wl.W).real)
        h0 = direct(wl.inj, f)
        d = wl.make_data(h0)
        h0e = direct(wl.inj, wl.f_edges)
        summ = orc.het_prepare(g.k_min, g.df, d, wl.W, h0, wl.f_edges)
        work = lambda n: orc.het_batch_standin(wl.modes_m, wl.c_lm, wl.kappa, wl.params[:n], wl.f_edges, h0e, summ)
        n_total = min(wl.n_w, n_sample or wl.n_w)
    return work, n_total, wl


def cpu_baseline(index: int, repeats: int = 3):
    """the oracle timed on this box's host cores: median of `repeats` runs on all cores (omp_get_max_threads) and on one
    core (a 1/cores share of the sample, so both legs take about as long)"""
    import oracle as orc
    work, n_all, wl = oracle_job(index)
    cores = orc.n_threads()

    def timed(n):
        ts = []
        for _ in range(repeats):
            t0 = time.perf_counter()
            work(n)
            ts.append(time.perf_counter() - t0)
        return statistics.median(ts)

    t_all = timed(n_all)
    n_one = max(1, n_all // cores)
    orc.set_threads(1)
    try:
        t_one = timed(n_one)
    finally:
        orc.set_threads(cores)
    what = "whole grid" if wl.path == "full" else "all %d bins" % (len(wl.f_edges) - 1)
    return {"value": n_all / t_all, "unit": UNIT, "cores": cores, "kind": "oracle", "median_of": repeats,
            "sample": f"{wl.name}: first {n_all} of {wl.n_w} walkers, {what}; {t_all:.2f} s per run on {cores} cores",
            "evals_per_s_all_cores": n_all / t_all, "evals_per_s_per_core": n_one / t_one,
            "per_core_sample": f"first {n_one} walkers on one thread, {t_one:.2f} s per run",
            "seconds": t_all, "n_sample": n_all}


def run_reference(args):
    """--impl reference: the oracle is the reference arm for this tier (no reference implementation exists).  Each
    step is the SAME bounded sample `cpu_baseline` times (config 2: the first CPU_SAMPLE_CFG2 walkers over the whole
    grid, on all cores), so the two legs agree."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle as orc
    orc.build()
    cores = orc.n_threads()
    work, n_sample, wl = oracle_job(args.workload)
    for _ in range(max(args.warmup, 0)):
        work(n_sample)
    ts = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        work(n_sample)
        ts.append(time.perf_counter() - t0)
    dt = sum(ts)
    val = n_sample * args.steps / dt
    what = "whole grid" if wl.path == "full" else "all bins"
    sample = f"{wl.name}: first {n_sample} of {wl.n_w} walkers per step, {what}"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 (x87 long double accumulators)", "data": "synthetic",
            "config": workload_config(wl),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                             "median_step_evals_per_s": n_sample / statistics.median(ts)},
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


def config_roofline(wl, ctx, kernel_ms: float, peak_slots: float):
    """ALU roofline of one configuration's dominant kernel: units of the launch x algorithmic FP64 slots per unit
    (SURVEY §8(d) for the formulation the kernel implements) / CUDA-event duration / peak"""
    if wl.path == "full":
        units = ctx.last_full_stats()[0]                # active (walker, bin, mode) triples, counted on the device
        if wl.n_m == 1:
            slots = SLOTS_FULL if wl.n_c == 2 else SLOTS_FULL_NC3
            out = {"kernel": "k_full_fused<1, %d, %s>" % (wl.n_c, "true" if wl.n_c == 2 else "false"), "slots_per_unit": slots,
                   "formulation": "rotation recurrence (SURVEY §8(d): ~27 for two channels), re-synchronised every 128 bins; "
                                  "the direct formulation needs %g" % SLOTS_FULL_DIRECT,
                   "frac_with_resync": units * (slots + SLOTS_RESYNC) / (kernel_ms * 1e-3) / peak_slots}
        else:
            slots = SLOTS_FULL_DIRECT
            out = {"kernel": "k_full_fused<0, %d, ...>" % wl.n_c, "slots_per_unit": slots, "formulation": "direct (SURVEY §8(d): 39)"}
        out["unit_name"] = "active (walker, bin, mode)"
    else:
        units = float(wl.n_w) * (len(wl.f_edges) - 1)
        slots = SLOTS_HET.get(wl.n_m, 73.0 + 36.0 * (wl.n_m - 1))
        out = {"kernel": "k_het_standin1" if wl.n_m == 1 else "k_het_standin<%d>" % wl.n_m, "slots_per_unit": slots,
               "unit_name": "(walker, bin)",
               "formulation": ("regrouped by edge (DESIGN.md §5): 48; the bin-by-bin form of SURVEY §8(d) needs %g"
                               % SLOTS_HET_SURVEY_FORM[1]) if wl.n_m == 1 else "bin by bin (SURVEY §8(d): 252 for six modes)"}
    out.update({"units": units, "kernel_ms": kernel_ms, "frac": units * slots / (kernel_ms * 1e-3) / peak_slots})
    return out


def sustained_dfma(torch, ctx, index: int, burst_ms_at_4000: float, seconds: float = 2.2):
    """the FP64 roofline denominator from a >= 2 s run of dependent-free DFMA chains on every SM, with the
    SM clock sampled during it (a burst of a few ms says nothing about the clock the chip holds under this load)"""
    iters = int(4000 * seconds * 1e3 / max(burst_ms_at_4000, 1e-3))
    with ClockSampler(index, period=0.05) as clk:
        rate, ms = ctx.peak_fma(0, iters)
    c = clk.summary()
    return {"measured_dfma_per_s_sustained": rate, "sustained_run_s": ms * 1e-3, "sustained_sm_mhz": c.get("sm_mhz"),
            "sustained_clock_reasons": c.get("reasons")}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", type=int, default=2, help="BASELINE.json config index of the headline step")
    ap.add_argument("--quick", action="store_true", help="skip per_config, e2e and cpu_baseline (profiling runs)")
    ap.add_argument("--n-walkers", type=int, default=None,
                    help="profiling aid: the headline workload with this many walkers (e.g. 160: one Module-1 sized call); "
                         "implies --quick, and the line's config says so")
    ap.add_argument("--channels", type=int, default=None, choices=[2, 3],
                    help="profiling aid: 3 = the headline workload with three channels and per-channel weight rows; implies --quick")
    ap.add_argument("--precision", default="fp64", choices=["fp64", "fp32acc"],
                    help="fp32acc: time the FP32-accumulate variant of the full-grid path as the headline step")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    if args.n_walkers is not None or args.channels == 3:
        args.quick = True

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
                           precision=1 if args.precision == "fp32acc" else 0, n_w=args.n_walkers, n_c=args.channels)
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
        k_ms = res["kernel_ms"]
        dfma_rate, dfma_ms = ctx.peak_fma(0, 4000)
        ffma_rate, _ = ctx.peak_fma(1, 8000)
        common = {"kernel_ms": k_ms, "kernel_share_of_step": k_ms / res["ms_per_step"],
                  "measured_dfma_per_s_burst": dfma_rate, "measured_ffma_per_s_burst": ffma_rate,
                  "hbm_peak_gbs": peaks.get("hbm_gbs"), "hbm_peak_source": peak_src}
        if not args.quick:
            common.update(sustained_dfma(torch, ctx, local, dfma_ms))
        if wl.path == "full" and args.precision == "fp32acc":
            pairs, n_blocks = ctx.last_full_stats()
            traffic, traffic_src = ncu_traffic_bytes("full_fused_mixed_cfg%d" % args.workload)
            peak_issue = n_sm * ISSUE_LANES_PER_CLK_PER_SM * sm_max * 1e6
            achieved = pairs * INSTR_FULL_FP32ACC / (k_ms * 1e-3)
            line["roofline"] = {
                "bound": "alu", "kernel": "k_full_fused_mixed", "achieved": achieved / 1e12, "peak": peak_issue / 1e12,
                "unit": "T lane-instructions/s (instruction issue: 1 warp instruction/scheduler/clk)",
                "frac": achieved / peak_issue, "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_instructions_per_pair": INSTR_FULL_FP32ACC, "active_pairs": pairs,
                "peak_source": f"{n_sm} SMs x 4 schedulers x 32 lanes x {sm_max:.0f} MHz (DESIGN.md §6)",
                "fp64_slots_per_pair": 13.0, "fp64_pipe_frac": pairs * 13.0 / (k_ms * 1e-3) / peak_slots, **common}
        else:
            rf = config_roofline(wl, ctx, k_ms, peak_slots)
            tag = ("full_fused_cfg%d" if wl.path == "full" else "het_cfg%d") % args.workload
            if args.n_walkers is not None:  # a capture belongs to one batch size: only the committed small-batch one applies
                tag = "small%d" % args.n_walkers
            elif args.channels == 3:
                tag += "_nc3"
            traffic, traffic_src = ncu_traffic_bytes(tag)
            line["roofline"] = {
                "bound": "alu", "kernel": rf["kernel"], "achieved": rf["frac"] * peak_slots / 1e12, "peak": peak_slots / 1e12,
                "unit": "T FP64 issue slots/s (1 DFMA|DMUL|DADD = 1 slot)", "frac": rf["frac"],
                "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_slots_per_unit": rf["slots_per_unit"], "units": rf["units"], "formulation": rf["formulation"],
                "peak_source": f"{n_sm} SMs x {int(DFMA_PER_CLK_PER_SM)} DFMA/clk x {sm_max:.0f} MHz (DESIGN.md §6)",
                "frac_of_measured_dfma_burst": rf["frac"] * peak_slots / dfma_rate, **common}
            if "frac_with_resync" in rf:
                line["roofline"]["frac_with_resync"] = rf["frac_with_resync"]
            if "measured_dfma_per_s_sustained" in common:
                line["roofline"]["frac_of_measured_dfma_sustained"] = rf["frac"] * peak_slots / common["measured_dfma_per_s_sustained"]

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
        # ---- every BASELINE.json config, device-resident, stand-in entry points, each with the ALU roofline of its
        # dominant kernel (library CUDA-event bracket) — configs 0 and 1 are launch-bound
        per = {}
        for idx in (0, 1, 2, 3, 4):
            key = f"cfg{idx}"
            if idx == args.workload:
                per[key] = {"evals_per_s": value, "ms_per_batch": t_ms / args.steps, "n_walkers": wl.n_w}
                if args.precision == "fp64":
                    rf = line["roofline"]
                    per[key].update({"kernel": rf["kernel"], "kernel_ms": rf["kernel_ms"], "slots_per_unit": rf["algorithmic_slots_per_unit"],
                                     "units": rf["units"], "frac": rf["frac"], "launch_bound": False, "covered_by": COVERED_BY[key]})
                continue
            st = 50 if idx != 2 else args.steps
            r = bench_config(torch, idx, st, 5, profile=True)
            rf = config_roofline(r["wl"], r["ctx"], r["kernel_ms"], peak_slots)
            per[key] = {"evals_per_s": r["wl"].n_w / (r["ms_per_step"] * 1e-3), "ms_per_batch": r["ms_per_step"],
                        "n_walkers": r["wl"].n_w, "launches_per_batch": r["launches"] / st, "kernel": rf["kernel"],
                        "kernel_ms": rf["kernel_ms"], "slots_per_unit": rf["slots_per_unit"], "units": rf["units"],
                        "unit": rf["unit_name"], "frac": rf["frac"], "formulation": rf["formulation"],
                        "launch_bound": idx in (0, 1), "covered_by": COVERED_BY[key]}
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
                    per[key].update({"ms_per_batch_graph": ms_g, "evals_per_s_graph": r["wl"].n_w / (ms_g * 1e-3)})
                    del gr
                except Exception as e:
                    per[key]["graph_error"] = repr(e)[:200]
            if idx == 1:
                # ---- the reference update inside the loop (every 5000 iterations)
                # and the brute-force audit of the heterodyned values, config-1 size
                c1, p1, n_e = r["ctx"], r["bufs"]["params"], len(r["wl"].f_edges)
                het = [x.clone() for x in c1.het_batch_standin(p1)]
                o1 = tuple(torch.empty_like(het[0]) for _ in range(3))
                ms_a = time_steps(torch, lambda: c1.het_audit_standin(p1, out=o1), 5, 2) / 5
                err = (het[0] - o1[0]).abs()
                below = o1[0].max() - o1[0]                # distance from the best dense log L of the population
                near = below < 50.0
                per["cfg1_audit"] = {"evals_per_s": r["wl"].n_w / (ms_a * 1e-3), "ms_per_batch": ms_a, "n_walkers": r["wl"].n_w,
                                     "max_abs_het_minus_dense_logL": float(err.max()), "median_abs_het_minus_dense_logL": float(err.median()),
                                     "dense_logL_range": [float(o1[0].min()), float(o1[0].max())],
                                     "n_within_50_of_best": int(near.sum()),
                                     "max_abs_err_within_50_of_best": float(err[near].max()) if bool(near.any()) else None,
                                     "max_rel_err_to_distance_from_best": float((err / below.clamp_min(1.0)).max()),
                                     "entry": "ll_het_audit_standin (direct template at every dense bin of the band)"}
                t0 = time.perf_counter()
                for _ in range(5):
                    c1.het_refresh_standin(p1, r["out"][0], n_e)          # synchronises the stream itself
                ms_ref = (time.perf_counter() - t0) / 5 * 1e3
                per["cfg1_refresh"] = {"ms_per_update": ms_ref, "n_edges": n_e, "n_f": r["wl"].grid.n_f,
                                       "entry": "ll_het_refresh_standin (argmax, h0 on the grid and at the edges, H0; host wall time, the call synchronises)"}
                per["module2_iteration"] = bench_sampler_iteration(torch, c1, r["wl"], p1)
                per["module2_iteration"]["covered_by"] = COVERED_BY["module2_iteration"]
            r["ctx"].destroy()
            del r
            torch.cuda.empty_cache()
        if args.workload == 2 and args.precision == "fp64":
            # ---- config 2's FP32-accumulate variant on the same data: throughput and its distance from FP64
            r = bench_config(torch, 2, args.steps, 5, profile=True, precision=1)
            dl = (r["out"][0] - headline_logL).abs()
            pairs_m = r["ctx"].last_full_stats()[0]
            per["cfg2_fp32acc"] = {"evals_per_s": r["wl"].n_w / (r["ms_per_step"] * 1e-3), "ms_per_batch": r["ms_per_step"],
                                   "n_walkers": r["wl"].n_w, "kernel": "k_full_fused_mixed", "kernel_ms": r["kernel_ms"],
                                   "max_abs_dlogL_vs_fp64": float(dl.max()), "rms_dlogL_vs_fp64": float(dl.pow(2).mean().sqrt()),
                                   "fp64_slots_per_unit": 13.0, "fp64_pipe_frac": pairs_m * 13.0 / (r["kernel_ms"] * 1e-3) / peak_slots,
                                   "covered_by": COVERED_BY["cfg2_fp32acc"]}
            r["ctx"].destroy()
            del r
            torch.cuda.empty_cache()
            # ---- config 2 with three channels (A, E, T; per-channel PSDs: SURVEY §8(f) item 1)
            from paper_2111_01064_b200 import synth
            wl3 = wlm.make_workload(2, n_c=3)
            c3 = synth.make_context(wl3)
            b3 = synth.setup(c3, wl3)
            o3 = tuple(torch.empty(wl3.n_w, dtype=torch.float64, device="cuda") for _ in range(3))
            fn = lambda: c3.full_batch_standin(wl3.f_nodes, b3["params"], out=o3)
            fn()
            c3.profile_enable(True)
            nst = max(args.steps // 2, 3)
            ms = time_steps(torch, fn, nst, 3) / nst
            kms, kn = c3.profile_read()
            c3.profile_enable(False)
            rf = config_roofline(wl3, c3, kms / max(kn, 1), peak_slots)
            per["cfg2_nc3"] = {"evals_per_s": wl3.n_w / (ms * 1e-3), "ms_per_batch": ms, "n_walkers": wl3.n_w, "n_channels": 3,
                               "kernel": rf["kernel"], "kernel_ms": rf["kernel_ms"], "slots_per_unit": rf["slots_per_unit"],
                               "units": rf["units"], "frac": rf["frac"], "frac_with_resync": rf["frac_with_resync"],
                               "entry": "ll_set_data(w_shared = 0), W [3][n_f]; ll_full_batch_standin with 11-double rows",
                               "covered_by": COVERED_BY["cfg2_nc3"]}
            c3.destroy()
            del b3, o3
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
                              "kernel": "k_full_fused_tf<1, 2, true>", "kernel_ms": kms / max(kn, 1), "units": pairs2,
                              "slots_per_unit": SLOTS_FULL_TF,
                              "frac": pairs2 * SLOTS_FULL_TF / (kms / max(kn, 1) * 1e-3) / peak_slots,
                              "entry": "ll_full_batch_tf (amp, phase, T at 1024 nodes as device arrays; the walkers' own bands)",
                              "covered_by": COVERED_BY["cfg2_tf"]}
            # the same entry point at Module-1 size (160 walkers: one-warp blocks over the planner's group items)
            a16, p16, t16, b16 = (v[:160].contiguous() for v in (amp, ph, tfn, bnd))
            o16 = tuple(torch.empty(160, dtype=torch.float64, device=amp.device) for _ in range(3))
            fn16 = lambda: c2.full_batch_tf(wl2.f_nodes, a16, p16, t16, band=b16, out=o16)
            fn16()
            c2.profile_enable(True)
            ms16 = time_steps(torch, fn16, 20, 3) / 20
            kms16, kn16 = c2.profile_read()
            c2.profile_enable(False)
            pairs16 = c2.last_full_stats()[0]
            per["cfg2_tf"]["call_160"] = {"n_walkers": 160, "ms_per_batch": ms16, "kernel_ms": kms16 / max(kn16, 1), "units": pairs16,
                                          "slots_per_unit": SLOTS_FULL_TF,
                                          "frac": pairs16 * SLOTS_FULL_TF / (kms16 / max(kn16, 1) * 1e-3) / peak_slots,
                                          "covered_by": "tests/test_parity_cfg2_scale.py::test_small_batch_tf_against_oracle"}
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
                              "kernel": "k_full_fused_pw<1, 2, true>", "kernel_ms": kms3 / max(kn3, 1), "units": pairs2,
                              "frac": pairs2 * SLOTS_FULL_PW / (kms3 / max(kn3, 1) * 1e-3) / peak_slots,
                              "slots_per_unit": SLOTS_FULL_PW,
                              "max_abs_dlogL_vs_shared_nodes": float((o3[0] - sh[0]).abs().max()),
                              "entry": "ll_full_batch_pw (f_nodes_w [n_w][1024] on the device; the walkers' own bands)",
                              "covered_by": COVERED_BY["cfg2_pw"]}
            # the same entry point at Module-1 size (block spline with a warm-up for the elimination factors, work items)
            x16, a16, p16, t16, b16 = (v[:160].contiguous() for v in (xw, amp, ph, tfc, bnd))
            o16 = tuple(torch.empty(160, dtype=torch.float64, device=amp.device) for _ in range(3))
            fn16 = lambda: c2.full_batch_pw(x16, a16, p16, t16, band=b16, out=o16)
            fn16()
            c2.profile_enable(True)
            ms16 = time_steps(torch, fn16, 20, 3) / 20
            kms16, kn16 = c2.profile_read()
            c2.profile_enable(False)
            pairs16 = c2.last_full_stats()[0]
            per["cfg2_pw"]["call_160"] = {"n_walkers": 160, "ms_per_batch": ms16, "kernel_ms": kms16 / max(kn16, 1), "units": pairs16,
                                          "slots_per_unit": SLOTS_FULL_PW,
                                          "frac": pairs16 * SLOTS_FULL_PW / (kms16 / max(kn16, 1) * 1e-3) / peak_slots,
                                          "covered_by": "tests/test_parity_cfg2_scale.py::test_small_batch_pw_against_oracle"}
            del xw, sh, tfc
            # ---- SURVEY §8(f) item 2, t_shift: the stand-in's linear phase term 2 pi f t_c kept outside the spline
            c2.standin_split_tc(True)
            o4 = tuple(torch.empty(wl2.n_w, dtype=torch.float64, device=amp.device) for _ in range(3))
            fn4 = lambda: c2.full_batch_standin(wl2.f_nodes, b2["params"], out=o4)
            fn4()
            c2.profile_enable(True)
            ms4 = time_steps(torch, fn4, nst, 2) / nst
            kms4, kn4 = c2.profile_read()
            c2.profile_enable(False)
            c2.standin_split_tc(False)
            dsp = (o4[0] - headline_logL).abs()
            per["cfg2_split_tc"] = {"evals_per_s": wl2.n_w / (ms4 * 1e-3), "ms_per_batch": ms4, "kernel_ms": kms4 / max(kn4, 1),
                                    "max_abs_dlogL_vs_full_phase_spline": float(dsp.max()),
                                    "max_abs_node_phase_rad": {"full": float(ph.abs().max()), "split": float((ph - 2 * np.pi * torch.as_tensor(wl2.f_nodes, device=ph.device) * b2["params"][:, 2:3, None]).abs().max())},
                                    "entry": "ll_standin_split_tc(1); ll_full_batch_standin (reading R32)",
                                    "covered_by": COVERED_BY["cfg2_split_tc"]}
            # ---- six modes through the full-grid path (the paper's higher-mode run used the brute-force likelihood)
            hm = bench_full_hm(torch)
            hm["frac"] = hm["active_pair_modes"] * hm["algorithmic_slots_per_pair_mode"] / (hm["kernel_ms"] * 1e-3) / peak_slots
            hm["covered_by"] = COVERED_BY["cfg2_hm6"]
            h16 = bench_full_hm(torch, steps=10, n_w=160)   # the same at Module-1 size: the kernel's item form on the small-batch route
            hm["call_160"] = {"n_walkers": 160, "ms_per_batch": h16["ms_per_batch"], "kernel_ms": h16["kernel_ms"],
                              "units": h16["active_pair_modes"], "slots_per_unit": h16["algorithmic_slots_per_pair_mode"],
                              "frac": h16["active_pair_modes"] * h16["algorithmic_slots_per_pair_mode"] / (h16["kernel_ms"] * 1e-3) / peak_slots}
            per["cfg2_hm6"] = hm
            # ---- Module-1 sized sampler iteration on the full-grid likelihood of the same one-year data stream
            per["module1_iteration"] = bench_sampler_iteration(torch, c2, wl2, b2["params"], n_t=4, n_w=80, iters=20,
                                                               f_nodes=wl2.f_nodes)
            per["module1_iteration"]["covered_by"] = COVERED_BY["module1_iteration"]
            per["module1_iteration"].update(bench_small_batch(torch, c2, wl2, b2["params"], peak_slots))
            # ---- the same likelihood call over the batch sizes between Module 1's and config 2's (first n walkers of config 2):
            # the small-batch route up to 1024 walkers, the large-batch route above
            sizes = {}
            for n in (37, 320, 1024, 2048, 4096):
                sizes.update(bench_small_batch(torch, c2, wl2, b2["params"], peak_slots, n_w=n, steps=10))
            sizes["covered_by"] = "tests/test_parity_cfg2_scale.py::test_module1_sized_batches_against_oracle (37 ... 2048), test_cfg2_full_size_128_walkers"
            per["cfg2_batch_sizes"] = sizes
            c2.destroy()
            del amp, ph, tfn, b2
            torch.cuda.empty_cache()
        line["per_config"] = per
        # ---- the oracle on this box's cores: the headline config, then every other config (het configs in full,
        # config 2 on a bounded sample), median of 3, per core and on all cores (SURVEY §8(d) "Oracle timing")
        import oracle as orc
        orc.build()
        cb = cpu_baseline(args.workload)
        cb["per_config"] = {f"cfg{i}": (cpu_baseline(i) if i != args.workload else "the headline entry above") for i in range(5)}
        line["cpu_baseline"] = cb
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
