"""Build the in-tree native libraries for sm_100a with nvcc (no torch extension machinery).

    python -m paper_2606_00516_b200.build            # build if stale
    python -m paper_2606_00516_b200.build --force

Outputs (git-ignored, shipped to the GPU box by gpurun):
    paper_2606_00516_b200/libpa_b200.so        the product: C ABI of include/pa.h
    paper_2606_00516_b200/synth/libpa_synth.so seeded input generator (device twin of synth/gen.py)
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpa_b200.so")
SYNTH_SRC = os.path.join(HERE, "synth", "synth_fill.cu")
SYNTH_LIB = os.path.join(HERE, "synth", "libpa_synth.so")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-shared", "--expt-relaxed-constexpr"]


def _stale(target: str, sources: list[str]) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def _run(cmd: list[str]) -> None:
    print("+", " ".join(cmd), flush=True)
    subprocess.check_call(cmd)


def build(force: bool = False, verbose_ptxas: bool = False) -> None:
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    deps = srcs + glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h")) + \
        [os.path.join(ROOT, "include", "pa.h")]
    extra = ["-Xptxas", "-v"] if verbose_ptxas else []
    if force or _stale(LIB, deps):
        tmp = LIB + f".{os.getpid()}.tmp"
        _run([NVCC, *ARCH, *COMMON, *extra, "-I", os.path.join(ROOT, "include"), "-o", tmp, *srcs])
        os.replace(tmp, LIB)
    if force or _stale(SYNTH_LIB, [SYNTH_SRC]):
        tmp = SYNTH_LIB + f".{os.getpid()}.tmp"
        _run([NVCC, *ARCH, *COMMON, "-o", tmp, SYNTH_SRC])
        os.replace(tmp, SYNTH_LIB)


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose_ptxas="-v" in sys.argv)
