"""Build libtcw.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2507_07816_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the
repository snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
# TCW_LIBRARY: build / load the library at another path (e.g. a variant built with TCW_NVCC_FLAGS="-DTCW_RB=2")
LIB = os.environ.get("TCW_LIBRARY") or os.path.join(HERE, "libtcw.so")
SOURCES = ["tcw_api.cu"]
DEPENDS = ["tcw_api.cu", "tcw_sum.cuh", "tcw_tables.cuh", "tcw_skyblock.cuh", "tcw_skyblock2.cuh", "tcw_bank.cuh", "tcw_select.cuh", "tcw_prep.cuh", "tcw_peaks.cuh", "tcw_exp_tables.inc", "tcw_pow_tables.inc", os.path.join("..", "..", "include", "tcw.h")]
NVCC_FLAGS = [
    "-O3", "-std=c++17",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo",
    "-fmad=false",            # bin indices are chains of single IEEE-754 operations: never contract
    "-Xcompiler", "-fPIC", "-shared",
    # cuFFT: the batched real-to-complex transform of tcw_prepare (a library primitive)
    "-lcufft", "-Xlinker", "-rpath", "-Xlinker", "/usr/local/cuda/lib64",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _flags() -> list[str]:
    return [*NVCC_FLAGS, *os.environ.get("TCW_NVCC_FLAGS", "").split()]


def _stamp_path() -> str:
    return LIB + ".flags"


def needs_build() -> bool:
    """True when the library is missing, older than a source, or was built with other nvcc flags
    (TCW_NVCC_FLAGS variants: the flag string is kept in a stamp file beside the library, so a
    variant measurement can never silently time a build made with different flags)."""
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    if any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPENDS):
        return True
    try:
        with open(_stamp_path()) as f:
            return f.read() != " ".join(_flags())
    except OSError:
        # no stamp (a library built before stamps existed): trust it only for the default flags
        return bool(os.environ.get("TCW_NVCC_FLAGS", "").split())


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        cmd = [_nvcc(), *_flags(), *(["-Xptxas", "-v"] if verbose else []),
               "-o", LIB, *[os.path.join(CSRC, s) for s in SOURCES]]
        subprocess.run(cmd, check=True)
        with open(_stamp_path(), "w") as f:
            f.write(" ".join(_flags()))
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
