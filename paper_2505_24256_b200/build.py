"""Build libzippel.so (the C-ABI CUDA library, include/zippel.h) in-tree with nvcc for sm_100a.

    python -m paper_2505_24256_b200.build [--force] [--verbose]

The .so is git-ignored but travels to the GPU box with the gpurun snapshot.  nvcc cross-compiles
without a GPU.  Nothing here falls back to anything: no nvcc -> the build raises.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
SO_PATH = os.path.join(_HERE, "libzippel.so")
SOURCES = [os.path.join(_CSRC, "zippel_capi.cu")]
HEADERS = [os.path.join(_CSRC, h) for h in ("modarith.cuh", "kernels.cuh")] + [
    os.path.join(os.path.dirname(_HERE), "include", "zippel.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "--shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libzippel.so cannot be built (there is no CPU fallback)")


def is_stale() -> bool:
    if not os.path.exists(SO_PATH):
        return True
    so_t = os.path.getmtime(SO_PATH)
    return any(os.path.getmtime(s) > so_t for s in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/zippel_capi.cu -> libzippel.so if missing or older than its sources."""
    if not (force or is_stale()):
        return SO_PATH
    tmp = SO_PATH + f".{os.getpid()}.tmp"
    cmd = [_nvcc()] + NVCC_FLAGS + ["-o", tmp] + SOURCES
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout)
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    os.replace(tmp, SO_PATH)
    log = os.path.join(_HERE, "csrc", "ptxas.log")
    with open(log, "w") as fh:
        fh.write(" ".join(cmd) + "\n" + res.stdout)
    if verbose:
        sys.stdout.write(res.stdout)
    return SO_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
