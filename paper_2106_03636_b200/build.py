"""In-tree build of libtpc_b200.so (hand-written CUDA for sm_100a behind the C ABI of include/tpc_b200.h).

`python -m paper_2106_03636_b200.build` or `build_library()`; nvcc cross-compiles without a GPU.
Flags that are part of the arithmetic contract: `-fmad=false` (one IEEE rounding per written
fp32 operation on the device; the fused multiply-adds of the contract are explicit __fmaf_rn) and
`-ffp-contract=off` for the host-side geometry tables.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtpc_b200.so")
SOURCES = ["tpc_api.cu", "tpc_grid.cu", "tpc_find.cu", "tpc_follow.cu", "tpc_select.cu", "tpc_fit.cu", "tpc_vertex.cu", "tpc_collisions.cu", "tpc_merge.cu", "tpc_cluster.cu"]
HEADERS = ["tpc_common.cuh", "tpc_kalman.cuh", "tpc_scan.cuh", "tpc_search.cuh", "tpc_prof.cuh", os.path.join("..", "..", "include", "tpc_b200.h")]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libtpc_b200.so cannot be built (there is no CPU fallback)")


def up_to_date() -> bool:
    if not os.path.exists(LIB):
        return False
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return all(os.path.getmtime(d) <= t for d in deps)


def build_library(force: bool = False, verbose: bool = False, out: str | None = None) -> str:
    """Compile csrc/*.cu -> paper_2106_03636_b200/libtpc_b200.so (or `out`) for sm_100a."""
    if out is None and not force and up_to_date():
        return LIB
    target = out or LIB
    tmp = target + f".tmp{os.getpid()}"
    cmd = [_nvcc(), "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-fmad=false",
           "-Xcompiler", "-fPIC,-ffp-contract=off", "-shared", "-o", tmp]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building libtpc_b200.so")
    os.replace(tmp, target)
    return target


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="-v" in sys.argv))
