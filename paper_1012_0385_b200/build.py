"""Build libkpz_b200.so (the product) and libkpz_b200_testhooks.so (test-only Philox dump kernel K0) in-tree
with nvcc for sm_100a.

Usage:  python -m paper_1012_0385_b200.build [--force]
nvcc cross-compiles without a GPU.  The built .so files are git-ignored but travel with the snapshot to the GPU box.
"""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
ROOT = os.path.dirname(HERE)
LIB = os.path.join(HERE, "libkpz_b200.so")
HOOKS = os.path.join(HERE, "libkpz_b200_testhooks.so")

NVCC = os.environ.get("NVCC", "nvcc")
FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]

LIB_SOURCES = ["kpz_api.cu", "lanes_api.cu"]
HOOK_SOURCES = ["testhooks.cu"]


def _deps():
    out = [os.path.join(ROOT, "include", "kpz_b200.h")]
    for f in sorted(os.listdir(CSRC)):
        if f.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, f))
    return out


def _stale(target: str) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(f) > t for f in _deps())


def _compile(src: str, extra=()) -> str:
    obj = os.path.join(CSRC, os.path.splitext(src)[0] + ".o")
    cmd = [NVCC, *FLAGS, *extra, "-c", os.path.join(CSRC, src), "-o", obj]
    subprocess.run(cmd, check=True, cwd=CSRC)
    return obj


def _link(objs, target):
    tmp = target + f".tmp{os.getpid()}"
    subprocess.run([NVCC, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", tmp, *objs], check=True, cwd=CSRC)
    os.replace(tmp, target)


def build(force: bool = False, verbose: bool = False) -> str:
    if not (force or _stale(LIB) or _stale(HOOKS)):
        return LIB
    extra = ["-Xptxas", "-v"] if verbose else []
    with cf.ThreadPoolExecutor(max_workers=4) as ex:
        futs = {s: ex.submit(_compile, s, extra) for s in LIB_SOURCES + HOOK_SOURCES}
        objs = {s: f.result() for s, f in futs.items()}
    _link([objs[s] for s in LIB_SOURCES], LIB)
    _link([objs[s] for s in HOOK_SOURCES], HOOKS)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
