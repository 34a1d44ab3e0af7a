"""Compile libscatman.so (sm_100a only) in-tree with nvcc.  No torch involved: the library is plain C ABI.

Every translation unit is compiled to an object under csrc/build/ (in parallel, only when it or a header is newer), then
linked; `python -m paper_2202_03411_b200.build [-v]` forces a full rebuild (-v adds -Xptxas -v)."""
from __future__ import annotations

import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libscatman.so")
SOURCES = ["api.cu", "fit_kernels.cu", "nufft_kernels.cu", "nufft_tensor_kernels.cu", "prep_kernels.cu", "render_kernels.cu",
           "sep_kernels.cu", "sep_tensor_kernels.cu", "simt_kernels.cu", "tensor_kernel.cu"]
HEADERS = ["internal.h", "ptx_sm100.h", "tc_cgemm.cuh", os.path.join("..", "..", "include", "scatman.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17"]
# SCATMAN_CHECKED=1: the same library with device-side checks compiled in (mbarrier watchdog, bounds assertions before stores
# and TMA loads; csrc/ptx_sm100.h).  compute-sanitizer is not available on the GPU pool, so this is the build the sanitize
# subset of the tests runs on (profiles/r02_sanitizers.md).  Objects go to their own directory; the output is still LIB.
CHECKED = os.environ.get("SCATMAN_CHECKED", "") not in ("", "0")
if CHECKED:
    NVCC_FLAGS = NVCC_FLAGS + ["-DSCATMAN_CHECKED"]
    OBJ = os.path.join(CSRC, "build_checked")
STAMP = LIB + ".mode"                # which mode LIB was last linked in ("checked" / "normal"); travels with LIB


def _sources():
    return SOURCES


def _headers_mtime() -> float:
    return max(os.path.getmtime(os.path.join(CSRC, h)) for h in HEADERS)


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    if not os.path.exists(STAMP) or open(STAMP).read().strip() != ("checked" if CHECKED else "normal"):
        return True                  # LIB was linked in the other mode
    t = os.path.getmtime(LIB)
    return _headers_mtime() > t or any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in _sources())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    hdr = _headers_mtime()

    def compile_one(src: str) -> str:
        obj = os.path.join(OBJ, src[:-3] + ".o")
        path = os.path.join(CSRC, src)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(path), hdr):
            cmd = [nvcc, *NVCC_FLAGS, "-Xcompiler", "-fPIC", "-c", "-o", obj, path]
            if verbose:
                cmd += ["-Xptxas", "-v"]
            subprocess.run(cmd, check=True)
        return obj

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        objs = list(ex.map(compile_one, _sources()))
    subprocess.run([nvcc, *NVCC_FLAGS, "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "-o", LIB, *objs], check=True)
    with open(STAMP, "w") as f:
        f.write("checked\n" if CHECKED else "normal\n")
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
