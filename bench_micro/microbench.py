"""Build and run bench_micro/pipe_microbench.cu: the B200 issue rates behind the alu-pipe slot roofline.

    python bench_micro/microbench.py            # needs a GPU; prints cycles per step for every instruction mix
    python bench_micro/microbench.py --build    # compile only (no GPU needed)
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pipe_microbench.cu")
EXE = os.path.join(HERE, "pipe_microbench")


def build() -> str:
    if not os.path.exists(EXE) or os.path.getmtime(EXE) < os.path.getmtime(SRC):
        subprocess.run([os.environ.get("NVCC", "nvcc"), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a",
                        "-lineinfo", "-o", EXE, SRC], check=True)
    return EXE


def main() -> int:
    exe = build()
    if "--build" in sys.argv:
        print(exe)
        return 0
    return subprocess.run([exe]).returncode


if __name__ == "__main__":
    sys.exit(main())
