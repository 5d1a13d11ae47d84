"""Build the C-ABI CUDA libraries in-tree with nvcc for sm_100a.

    python -m paper_2505_24256_b200.build [--force] [--verbose]

  libzippel.so       the product (include/zippel.h)
  libzippel_test.so  the same sources compiled with -DZP_TEST_HOOKS: adds the self-test, micro-benchmark and
                     intermediate-stage hooks of include/zippel_test.h (tests/ and the ubench module load it)

The .so files are git-ignored but travel to the GPU box with the gpurun snapshot.  nvcc cross-compiles
without a GPU.  Nothing here falls back to anything: no nvcc -> the build raises.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_INC = os.path.join(os.path.dirname(_HERE), "include")
SO_PATH = os.path.join(_HERE, "libzippel.so")
TEST_SO_PATH = os.path.join(_HERE, "libzippel_test.so")
SOURCES = [os.path.join(_CSRC, "zippel_capi.cu")]
HEADERS = [os.path.join(_CSRC, h) for h in ("modarith.cuh", "kernels.cuh", "ntt.cuh", "subq.cuh", "small.cuh")] + [
    os.path.join(_INC, "zippel.h")]
TEST_HEADERS = HEADERS + [os.path.join(_CSRC, h) for h in ("ubench.cuh", "test_hooks.cuh")] + [
    os.path.join(_INC, "zippel_test.h")]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "--shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libzippel.so cannot be built (there is no CPU fallback)")


def _stale(so: str, deps) -> bool:
    if not os.path.exists(so):
        return True
    so_t = os.path.getmtime(so)
    return any(os.path.getmtime(s) > so_t for s in deps)


def is_stale() -> bool:
    return _stale(SO_PATH, SOURCES + HEADERS)


def test_is_stale() -> bool:
    return _stale(TEST_SO_PATH, SOURCES + TEST_HEADERS)


def _compile(so: str, extra, log_name: str, verbose: bool) -> str:
    tmp = so + f".{os.getpid()}.tmp"
    cmd = [_nvcc()] + NVCC_FLAGS + extra + ["-o", tmp] + SOURCES
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout)
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    os.replace(tmp, so)
    with open(os.path.join(_CSRC, log_name), "w") as fh:
        fh.write(" ".join(cmd) + "\n" + res.stdout)
    if verbose:
        sys.stdout.write(res.stdout)
    return so


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/zippel_capi.cu -> libzippel.so if missing or older than its sources."""
    if not (force or is_stale()):
        return SO_PATH
    return _compile(SO_PATH, [], "ptxas.log", verbose)


def build_test(force: bool = False, verbose: bool = False) -> str:
    """The same sources with -DZP_TEST_HOOKS -> libzippel_test.so."""
    if not (force or test_is_stale()):
        return TEST_SO_PATH
    return _compile(TEST_SO_PATH, ["-DZP_TEST_HOOKS"], "ptxas_test.log", verbose)


def build_all(force: bool = False, verbose: bool = False):
    with ThreadPoolExecutor(2) as ex:
        a, b = ex.submit(build, force, verbose), ex.submit(build_test, force, verbose)
        return a.result(), b.result()


if __name__ == "__main__":
    print(*build_all(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
