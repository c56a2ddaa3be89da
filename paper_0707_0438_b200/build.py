"""Build csrc/ into libnbk.so for sm_100a with nvcc (in-tree, so the .so travels with gpurun).

    python -m paper_0707_0438_b200.build [--force]

nvcc cross-compiles without a GPU.  The library links the static CUDA runtime, so it can be
loaded next to torch's own runtime; both use the device's primary context.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
INCLUDE = os.path.join(ROOT, "include")
SOURCES = ["nbk_force.cu", "nbk_state_kernels.cu", "nbk_batch_kernels.cu", "nbk_hermite_kernels.cu", "nbk_hermite_steps.cu", "nbk_small_kernels.cu", "nbk_shard_kernels.cu", "nbk_noalloc.cu", "nbk_api.cu",
           "nbk_hermite_dev.cu", "nbk_batch.cu", "nbk_hermite.cpp"]
HEADERS = [os.path.join(CSRC, h) for h in ("nbk_kernels.cuh", "nbk_device.cuh", "nbk_ctx.cuh", "nbk_hermite_common.h")] + [os.path.join(INCLUDE, "nbk.h")]
LIB = os.path.join(HERE, "libnbk.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC,-O2,-fvisibility=default,-fopenmp",
    "-shared", "-cudart", "static",
]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA path cannot be built (there is no CPU fallback)")


def is_stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, lib: str = LIB, defines=(), verbose: bool = False) -> str:
    if not force and not is_stale(lib):
        return lib
    cmd = [nvcc_path(), *NVCC_FLAGS, "-I", INCLUDE]
    cmd += [f"-D{d}" for d in defines]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-lgomp", "-o", lib]
    proc = subprocess.run(cmd, capture_output=True, text=True)
    if proc.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + proc.stdout + proc.stderr)
    if verbose:
        sys.stderr.write(proc.stderr)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
