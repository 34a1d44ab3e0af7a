"""Compile libscatman.so (sm_100a only) in-tree with nvcc.  No torch involved: the library is plain C ABI."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libscatman.so")
SOURCES = ["api.cu", "fit_kernels.cu", "nufft_kernels.cu", "prep_kernels.cu", "render_kernels.cu", "sep_kernels.cu", "sep_tensor_kernels.cu", "simt_kernels.cu", "tensor_kernel.cu"]
HEADERS = ["internal.h", "ptx_sm100.h", os.path.join("..", "..", "include", "scatman.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "--use_fast_math=false"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")]
    cmd = [nvcc, *flags, "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
