"""Build libu1mps.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2303_11409_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libu1mps.so")
SOURCES = ["api.cu", "plan.cu", "contract.cu", "svd.cu", "select.cu", "readout.cu", "envs.cu"]
PROBE = os.path.join(HERE, "fp64_probe")          # measured FP64 peak (csrc/fp64_probe.cu), run by bench.py
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--extended-lambda",
         "-shared", "-Xcompiler", "-fPIC"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "u1mps.h")]
    return any(os.path.getmtime(p) > t for p in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    extra = os.environ.get("U1MPS_NVCC_FLAGS", "").split()   # e.g. -DSV_PROFILE for an instrumented debug build
    cmd = [nvcc] + FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stdout + res.stderr)
    if verbose:
        print(res.stderr)
    res = subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", PROBE,
                          os.path.join(CSRC, "fp64_probe.cu")], capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed (fp64_probe):\n" + res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
