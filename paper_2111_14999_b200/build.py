"""Build the sm_100a C-ABI library in-tree: paper_2111_14999_b200/libphoebe_elph.so.

Usage: python -m paper_2111_14999_b200.build [--force] [--verbose]
nvcc cross-compiles for sm_100a without a GPU.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = os.path.join(HERE, "csrc", "phoebe_elph.cu")
LIB = os.path.join(HERE, "libphoebe_elph.so")


def _deps():
    return (glob.glob(os.path.join(HERE, "csrc", "*.cu")) + glob.glob(os.path.join(HERE, "csrc", "*.cuh"))
            + glob.glob(os.path.join(ROOT, "include", "*.h")))


def nvcc_cmd(verbose: bool = False):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC",
           "-o", LIB, SRC]
    extra = os.environ.get("PHOEBE_ELPH_NVCC_FLAGS", "").split()      # e.g. -D switches of kernel experiments
    cmd[1:1] = extra
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    return cmd


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps()):
        return LIB
    subprocess.run(nvcc_cmd(verbose), check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
