"""Build the CPU oracle (test infrastructure) into oracle/libkpz_oracle.so with gcc.

Usage:  python -m oracle.build      (also called by __graft_entry__.build and by oracle/kpzref.py on demand)
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "kpz_oracle.c")
HDR = os.path.join(HERE, "kpz_oracle.h")
LIB = os.path.join(HERE, "libkpz_oracle.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in (SRC, HDR))


def build(force: bool = False) -> str:
    if force or needs_build():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = ["gcc", "-std=c11", "-O3", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=HERE)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
