"""In-tree build of the C-ABI CUDA library for sm_100a (nvcc, no torch involved).

    python -m paper_1011_4687_b200.build [--force] [--verbose]

Produces paper_1011_4687_b200/libqmmm_field.so next to this file (git-ignored; it
travels to the GPU box with the snapshot).  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libqmmm_field.so")
SOURCES = ["qmmm_field.cu", "qmmm_probe.cu", "qmmm_noalloc.cu"]
HEADERS = [os.path.join(CSRC, "qmmm_kernels.cuh"), os.path.join(CSRC, "qmmm_grid.cuh"),
           os.path.join(CSRC, "qmmm_server.cuh"),
           os.path.join(os.path.dirname(HERE), "include", "qmmm_field.h")]
# No --use_fast_math: the approximate instructions the kernels want are called
# explicitly.  -lineinfo keeps ncu's source page usable.
NVCC_FLAGS = ["-O3", "-std=c++17", "-lineinfo",
              "-gencode", "arch=compute_100a,code=sm_100a",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, defines=(), out: str = LIB) -> str:
    """Compile the library.  ``defines`` (e.g. ["QMMM_BLOCK_CHUNKS=8"]) and ``out`` build a
    tuning variant elsewhere; load it with the QMMM_FIELD_LIB environment variable."""
    if out == LIB and not defines and not force and not is_stale():
        return LIB
    cmd = [_nvcc(), *NVCC_FLAGS, *[f"-D{d}" for d in defines]]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-o", out]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libqmmm_field.so")
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
