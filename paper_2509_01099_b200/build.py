"""Build step: nvcc -> paper_2509_01099_b200/libislbm.so (sm_100a, in-tree)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libislbm.so")
SOURCES = ["islbm_api.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "--compiler-options", "-fPIC", "-shared",
]


def _deps():
    out = [os.path.join(HERE, "..", "include", "islbm.h")]
    for fn in os.listdir(CSRC):
        if fn.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, fn))
    return out


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in _deps())


def build(force: bool = False, verbose: bool = False) -> str:
    if force or is_stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        tmp = LIB + f".tmp{os.getpid()}"
        # ISLBM_NVCC_FLAGS: extra flags for A/B builds of the compile-time variants, e.g. -DISLBM_G_FP32=0 (profiles/attempts.md)
        extra = os.environ.get("ISLBM_NVCC_FLAGS", "").split()
        cmd = [nvcc, *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *SOURCES]
        subprocess.run(cmd, check=True, cwd=CSRC)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
