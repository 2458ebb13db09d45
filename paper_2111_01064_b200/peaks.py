"""Measured ALU peaks of this GPU through the library's own microbenchmark kernels (`ll_peak_fma`).

    python -m paper_2111_01064_b200.peaks

Prints one line per pattern: FMA/s and FMA per clock per SM at the SM's maximum clock.  These are the
denominators DESIGN.md §6 derives the ALU roofline from (the unit count 64 DFMA/clk/SM) and the evidence for
the operand-pattern ceiling of the fused kernel (profiles/).
"""
from __future__ import annotations

import torch

from .binding import Context

PATTERNS = ((0, "DFMA  a = fma(a, m, c), m and c loop-invariant registers", 4000),
            (2, "DFMA  three distinct register operands", 4000),
            (3, "DFMA  one operand from the constant bank", 4000),
            (4, "DFMA  constant bank + 1 integer add per 2 DFMA", 4000),
            (5, "DFMA  constant bank + 1 integer add per DFMA", 4000),
            (6, "DFMA  constant bank + 1 FFMA per 2 DFMA", 4000),
            (7, "DFMA  constant bank + 1 FFMA per DFMA", 4000),
            (1, "FFMA  a = fma(a, m, c)", 8000))


def main() -> int:
    if not torch.cuda.is_available():
        raise SystemExit("peaks: no CUDA device")
    props = torch.cuda.get_device_properties(0)
    try:
        import pynvml
        pynvml.nvmlInit()
        mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(pynvml.nvmlDeviceGetHandleByIndex(0), pynvml.NVML_CLOCK_SM))
    except Exception:
        mhz = 1965.0
    ctx = Context(n_modes=1)
    print(f"{props.name}: {props.multi_processor_count} SMs, SM max clock {mhz:.0f} MHz")
    for which, label, iters in PATTERNS:
        rate, ms = ctx.peak_fma(which, iters)
        print(f"{label:62s} {rate / 1e12:7.2f} T/s  {rate / props.multi_processor_count / (mhz * 1e6):6.1f} /clk/SM  ({ms:.2f} ms)")
    ctx.destroy()
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
