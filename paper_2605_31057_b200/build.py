"""Builds csrc/*.cu into csrc/liblvsa.so with nvcc for sm_100a (in-tree, so the .so travels
to the GPU box with the repo snapshot)."""
from __future__ import annotations

import glob
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(CSRC, "liblvsa.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "-Xptxas", "-v"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = sources() + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) \
        + glob.glob(os.path.join(INCLUDE, "*.h"))
    return any(os.path.getmtime(d) > t for d in deps)


NVCC = "/usr/local/cuda/bin/nvcc"


def _compile(out: str, extra_flags=(), verbose: bool = False):
    cmd = [NVCC, *NVCC_FLAGS, *extra_flags, "-I", INCLUDE, "-I", CSRC, "-o", out, *sources()]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        print(r.stdout)
        print(r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed building %s (see output above)" % os.path.basename(out))
    return cmd, r


def build(force: bool = False, verbose: bool = False) -> str:
    """The product library, rebuilt when a source is newer.  Always this path: nothing outside the call can substitute another library."""
    if not force and not stale():
        return LIB
    cmd, r = _compile(LIB, verbose=verbose)
    with open(os.path.join(CSRC, "build.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + r.stdout + r.stderr)
    return LIB


def build_variant(out: str, extra_flags) -> str:
    """A separate build of the same sources with extra nvcc flags, written to `out` (never the product
    path): the fault-injection test compiles one with -DLVSA_TEST_CAP_SHRINK (tests/test_gpu_overflow.py)."""
    if os.path.abspath(out) == os.path.abspath(LIB):
        raise ValueError("a variant build must not overwrite the product library")
    _compile(out, extra_flags=tuple(extra_flags))
    return out


if __name__ == "__main__":
    print(build(force=True, verbose=True))
