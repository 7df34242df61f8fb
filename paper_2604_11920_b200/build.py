"""Build libtomolsqr.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension machinery).

``python -m paper_2604_11920_b200.build`` or :func:`build`.  The flags matter for correctness:
``--fmad=false`` keeps the double-double error-free transformations and the scalar recurrences free of
FMA contraction (a fused multiply-add exists only where ``fma()`` is written).
"""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libtomolsqr.so")
SOURCES = ["tomo_lsqr.cu"]
HEADERS = ["accum.cuh", "state.cuh", "tails.cuh", "kernels.cuh", "wstream.cuh", "compress.cuh", "wspmm.cuh", "shard.cuh", "multi.cuh", "build.cuh", "factored.cuh", os.path.join("..", "..", "include", "tomo_lsqr.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "--fmad=false", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libtomolsqr.so cannot be built (there is no CPU fallback)")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB + ".tmp"]
    subprocess.run(cmd, check=True, cwd=CSRC)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
