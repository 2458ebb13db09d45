"""nvcc build of csrc/ into libll_b200.so, in-tree, sm_100a only (no other arch, no PTX fallback path).

`python -m paper_2111_01064_b200.build [--force] [--verbose]`
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libll_b200.so")
SOURCES = [os.path.join(CSRC, "ll_b200.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "ll_kernels.cuh"), os.path.join(CSRC, "ll_device.cuh"),
                  os.path.join(ROOT, "include", "ll.h")]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built (there is no CPU fallback)")


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return SO
    cmd = [nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(ROOT, "include"), "-I", CSRC,
           "-o", SO] + SOURCES
    cmd[1:1] = os.environ.get("LL_NVCC_FLAGS", "").split()  # e.g. -DLL_FUSED_UNROLL=4 for tuning sweeps
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
