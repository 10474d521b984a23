"""Builds libtpcgpu.so (hand-written CUDA for sm_100a) in-tree with nvcc.

Flags (R0): --fmad=false -prec-div=true -prec-sqrt=true -ftz=false: every fp32 operation of the
selection and Kalman arithmetic is rounded once, exactly as written.  -lineinfo keeps ncu's source page usable.
"""
from __future__ import annotations

import glob
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
LIB = os.path.join(_HERE, "libtpcgpu.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--fmad=false",
              "-prec-div=true", "-prec-sqrt=true", "-ftz=false", "-shared", "-Xcompiler", "-fPIC"]


def _sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) +
                  glob.glob(os.path.join(INCLUDE, "*.h")))


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in _sources())


def build_cuda(force: bool = False, verbose: bool = False, defines=(), out: str | None = None) -> str:
    """Compile csrc/tpc_api.cu (which includes every kernel header) and csrc/tpc_noalloc.cu (the allocation-free entry
    point, a translation unit of its own) into libtpcgpu.so.

    ``defines`` / ``out`` build a tuning variant (-DNAME=VALUE ...) under another file name; the product is
    always the default build.
    """
    if out is not None:
        nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
        subprocess.check_call([nvcc] + NVCC_FLAGS + [f"-D{d}" for d in defines] +
                              [os.path.join(CSRC, "tpc_api.cu"), os.path.join(CSRC, "tpc_noalloc.cu"), "-o", out])
        return out
    if not force and not is_stale():
        return LIB
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        raise RuntimeError("nvcc not found: libtpcgpu.so cannot be built (there is no CPU fallback)")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          [os.path.join(CSRC, "tpc_api.cu"), os.path.join(CSRC, "tpc_noalloc.cu"), "-o", LIB]
    subprocess.check_call(cmd)
    return LIB


def emit_ptx(out: str) -> str:
    """The PTX of every kernel under the product's own arithmetic flags (for tests/test_build_flags.py: R0 is a property
    of the generated code, not only of a command line)."""
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    flags = [f for f in NVCC_FLAGS if f not in ("-shared", "-Xcompiler", "-fPIC", "-lineinfo")]
    flags[flags.index("-gencode") + 1] = "arch=compute_100a,code=compute_100a"
    subprocess.check_call([nvcc] + flags + ["-ptx", os.path.join(CSRC, "tpc_api.cu"), "-o", out])
    return out


if __name__ == "__main__":
    print(build_cuda(force=True, verbose=True))
