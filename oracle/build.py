"""Compile oracle/msft_oracle.c into oracle/libmsft_oracle.so with gcc (no CUDA involved).

ORACLE_SANITIZE=1 builds libmsft_oracle_san.so with -fsanitize=address,undefined instead (SURVEY section 4 tier T5); run the CPU
pins against it with the sanitizer runtime preloaded:
    ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so):$(gcc -print-file-name=libubsan.so) \
        ASAN_OPTIONS=detect_leaks=0 UBSAN_OPTIONS=halt_on_error=1 python -m pytest tests -m "not gpu" -q
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "msft_oracle.c")
SANITIZE = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
LIB = os.path.join(HERE, "libmsft_oracle_san.so" if SANITIZE else "libmsft_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]
    if SANITIZE:
        cmd[1:2] = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer", "-fno-sanitize-recover=undefined"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
