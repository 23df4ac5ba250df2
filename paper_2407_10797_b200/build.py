"""Build step of the CUDA library: nvcc -> paper_2407_10797_b200/libfstat_b200.so (in-tree, sm_100a only).

Run as ``python -m paper_2407_10797_b200.build [--force] [--verbose]`` or call ``build()``.
nvcc cross-compiles without a GPU.  The shared object is git-ignored but travels with the tree.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libfstat_b200.so")
SOURCES = ("fstat_api.cu", "fstat_kernels.cu", "fstat_fast.cu", "fstat_fastmulti.cu", "fstat_fastband.cu", "fstat_pso.cu", "fstat_band.cu")
HEADERS = ("fstat_internal.h", "fstat_device.cuh", "fstat_model.cuh", "fstat_direct.cuh", "fstat_fast.cuh")


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.join(INCLUDE, "fstat.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def command(out: str, verbose: bool = False):
    cmd = [_nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-Xcompiler", "-fPIC,-fvisibility=hidden", "-shared", "-I", INCLUDE, "-o", out]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    return cmd + [os.path.join(CSRC, s) for s in SOURCES]


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the library if it is missing or older than its sources; return its path."""
    if not force and not _stale():
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = command(tmp, verbose)
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout)
    if r.returncode != 0:
        if os.path.exists(tmp):
            os.remove(tmp)
        raise RuntimeError("nvcc failed (%d): %s" % (r.returncode, " ".join(cmd)))
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
