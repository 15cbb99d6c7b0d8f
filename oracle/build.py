"""Build the CPU oracle (test infrastructure) into oracle/libkpz_oracle.so with gcc.

Usage:  python -m oracle.build               (also called by __graft_entry__.build and by oracle/kpzref.py on demand)
        python -m oracle.build --sanitize    same library with -fsanitize=address,undefined (-O1 -g): run the oracle pins
                                             under it with LD_PRELOAD=$(gcc -print-file-name=libasan.so), then rebuild
                                             with --force (profiles/r02_sanitizers.md holds the commands and the result)
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "kpz_oracle.c")
HDR = os.path.join(HERE, "kpz_oracle.h")
SRC2D = os.path.join(HERE, "kpz2d_oracle.c")   # the 2+1D generalisation (calls the exported RNG functions of kpz_oracle.c)
HDR2D = os.path.join(HERE, "kpz2d_oracle.h")
LIB = os.path.join(HERE, "libkpz_oracle.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in (SRC, HDR, SRC2D, HDR2D))


def build(force: bool = False, sanitize: bool = False) -> str:
    if force or sanitize or needs_build():
        tmp = LIB + f".tmp{os.getpid()}"
        opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"] if sanitize else ["-O3"]
        cmd = ["gcc", "-std=c11", *opt, "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, SRC, SRC2D, "-lm"]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, sanitize="--sanitize" in sys.argv))
