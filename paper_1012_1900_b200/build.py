"""Build step: nvcc-compile csrc/gamma_api.cu into libgamma_b200.so (sm_100a only), in-tree.

    python -m paper_1012_1900_b200.build [--force] [--verbose]

No JIT cache is used: the .so sits next to this file so that it travels with the source tree.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgamma_b200.so")
SOURCES = ["gamma_api.cu"]
DEPENDS = ["common.cuh", "features_generated.cuh", "gamma_search.cuh", "ju_simplex.cuh", "offset_table.cuh", "radix_sort.cuh",
           "stats.cuh", "tile_star.cuh", "general.cuh", "gen_features.py", os.path.join("..", "..", "include", "gamma_b200.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "--shared", "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
]


def _nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: libgamma_b200.so cannot be built (there is no CPU fallback)")
    return exe


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    files = [os.path.join(CSRC, s) for s in SOURCES + DEPENDS]
    return any(os.path.getmtime(f) > t for f in files)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if needed; returns the path of the shared library."""
    if not force and not is_stale():
        return LIB
    extra = os.environ.get("GAMMA_NVCC_EXTRA", "").split()     # e.g. -DGAMMA_STAR_MIN_BLOCKS=4 for tuning runs
    cmd = [_nvcc()] + NVCC_FLAGS + extra + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    log = res.stdout + res.stderr
    with open(os.path.join(HERE, "build.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + log)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + log)
    if verbose:
        print(log)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
