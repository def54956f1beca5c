"""Builds paper_1911_09340_b200/libcomet.so (sm_100a only) with nvcc, in-tree.

    python -m paper_1911_09340_b200.build [--force]
"""
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.path.join(_HERE, "libcomet.so")
_SOURCES = ["comet_api.cu"]
_DEPS = ["comet_api.cu", "common.cuh", "extrapolate.cuh", "dca.cuh", "select.cuh", "scan_fused.cuh",
         "refine.cuh", "turns.cuh", "hough.cuh", "half.cuh", "scan_zgroup.cuh", "scan_zrun.cuh", "scan_small.cuh", "seedgrid.cuh",
         os.path.join("..", "..", "include", "comet.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC,-ffp-contract=off", "--shared",
]


def _stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    t = os.path.getmtime(LIB_PATH)
    return any(os.path.getmtime(os.path.join(_CSRC, d)) > t for d in _DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB_PATH
    nvcc = os.environ.get("NVCC", "nvcc")
    extra = os.environ.get("COMET_NVCC_EXTRA", "").split()      # e.g. -DCOMET_PRUNED_WT=2 for tuning runs
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB_PATH] + \
          [os.path.join(_CSRC, s) for s in _SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if verbose:
        sys.stderr.write(r.stderr)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
