"""Builds libmcx_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libmcx_b200.so")
# Same sources with FMA contraction off: per-ray arithmetic is then rounded like the oracle's (g++ -ffp-contract=off)
# and only the libm-vs-CUDA math functions differ.  Used by the parity tests to tell rounding from bugs (reading R20).
LIB_STRICT = os.path.join(_HERE, "libmcx_b200_strict.so")
SOURCES = ["mcx_kernels.cu", "mcx_host.cu"]
HEADERS = [os.path.join(CSRC, "mcx_device.h"), os.path.join(_HERE, "..", "include", "mcx.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
              "-shared"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build(lib=LIB):
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False, strict=False):
    """Compile the CUDA library if it is missing or older than its sources.  Returns the path of the .so."""
    lib = LIB_STRICT if strict else LIB
    if not force and not needs_build(lib):
        return lib
    cmd = [_nvcc()] + NVCC_FLAGS + (["-fmad=false"] if strict else []) + (["-Xptxas", "-v"] if verbose else [])
    subprocess.check_call(cmd + ["-o", lib] + SOURCES, cwd=CSRC)
    return lib


def build_all(force=False):
    return [build(force=force), build(force=force, strict=True)]


if __name__ == "__main__":
    print(build(force=True, verbose=True))
    print(build(force=True, strict=True))
