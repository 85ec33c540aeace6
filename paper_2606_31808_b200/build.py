"""In-tree build of the C-ABI library (libcd.so) for sm_100a with nvcc.

    python -m paper_2606_31808_b200.build [--force] [--verbose] [--nvtx] [--tuning]

--nvtx / --tuning build a second library (libcd_nvtx.so / libcd_tuning.so) beside the product one:
NVTX ranges per loop and decoding step, and the environment knobs used by the launch-shape sweeps.

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.
nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libcd.so")
SOURCES = [os.path.join(CSRC, "cd_api.cu")]
DEPS = [os.path.join(CSRC, f) for f in ("cd_api.cu", "cd_step.cuh", "cd_head.cuh", "cd_dedup.cuh", "cd_types.hpp", "cd_aux.cuh", "cd_common.cuh")] + [
    os.path.join(ROOT, "include", "cd.h"), os.path.join(ROOT, "include", "cd_diag.h")
]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
    "-shared",
]


def nvcc_path() -> str:
    for p in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc"):
        if p and os.path.exists(p):
            return p
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False, defines=(), out: str = SO) -> str:
    """defines: extra -D flags.  CD_NVTX = NVTX ranges around every loop and decoding step;
    CD_TUNING = the environment knobs of the launch-shape sweeps (never set for the product .so).  A build
    with defines should go to another `out` path."""
    if not force and out == SO and not needs_build():
        return SO
    tmp = out + f".tmp{os.getpid()}"
    cmd = [nvcc_path()] + NVCC_FLAGS + [f"-D{d}" for d in defines] + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    subprocess.check_call(cmd)
    os.replace(tmp, out)
    return out


if __name__ == "__main__":
    defs = [d for f, d in (("--nvtx", "CD_NVTX"), ("--tuning", "CD_TUNING")) if f in sys.argv]
    target = SO if not defs else os.path.join(HERE, "libcd_" + "_".join(d[3:].lower() for d in defs) + ".so")
    print(build(force="--force" in sys.argv or bool(defs), verbose="--verbose" in sys.argv, defines=defs, out=target))
