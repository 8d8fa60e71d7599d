"""Builds libpdv_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2012_00963_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libpdv_b200.so")
SOURCES = ["pdv_optics.cpp", "pdv_kernels.cu", "pdv_api.cu"]
HEADERS = ["pdv_optics.hpp", "pdv_device.h", os.path.join("..", "..", "include", "pdv.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC,-O3", "-shared", "-cudart", "static"]


def kernel_source_hash() -> str:
    """sha256 over the sources of the CUDA kernels (csrc/pdv_kernels.cu, csrc/pdv_device.h): the key that ties an ncu capture
    under profiles/ to the kernel it was taken from (bench.py prints a capture's counters only when the key matches)."""
    import hashlib
    h = hashlib.sha256()
    for f in ("pdv_kernels.cu", "pdv_device.h"):
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, extra_flags=(), out: str | None = None) -> str:
    """Compile the CUDA library if a source is newer than the .so.  Returns the .so path.
    extra_flags / out: an experiment build (-D macros of csrc/) into another file; the product build passes neither."""
    if out is not None or force or needs_build():
        tmp = (out or LIB) + f".tmp{os.getpid()}"
        cmd = [_nvcc()] + NVCC_FLAGS + list(extra_flags) + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", tmp] + [os.path.join(CSRC, f) for f in SOURCES]
        subprocess.check_call(cmd)
        os.replace(tmp, out or LIB)
    return out or LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
