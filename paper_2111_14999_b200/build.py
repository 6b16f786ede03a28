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
PROBES_SRC = os.path.join(HERE, "csrc", "probes.cu")
PROBES_LIB = os.path.join(HERE, "libphoebe_elph_probes.so")      # measurement aids of bench.py, not the product


def _deps():
    return (glob.glob(os.path.join(HERE, "csrc", "*.cu")) + glob.glob(os.path.join(HERE, "csrc", "*.cuh"))
            + glob.glob(os.path.join(ROOT, "include", "*.h")))


OBJ_DIR = os.path.join(HERE, "build")
ROT3_SRC = os.path.join(HERE, "csrc", "rot3_instances.cu")
NOALLOC_SRC = os.path.join(HERE, "csrc", "noalloc.cu")       # phoebe_elph_set_k_noalloc: fixed device scratch, no workspace
ROT3_PARTS = 4


def _nvcc_base(verbose: bool = False):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC"]
    cmd[1:1] = os.environ.get("PHOEBE_ELPH_NVCC_FLAGS", "").split()      # e.g. -D switches of kernel experiments
    if verbose:
        cmd[1:1] = ["-Xptxas", "-v"]
    return cmd


def nvcc_cmds(verbose: bool = False):
    """-> (compile commands, link command): the C ABI + most kernels (phoebe_elph.cu) and the instantiations of the
    rotation kernel in ROT3_PARTS translation units, compiled in parallel, linked into one shared library."""
    base = _nvcc_base(verbose)
    objs = [os.path.join(OBJ_DIR, "phoebe_elph.o")] + [os.path.join(OBJ_DIR, "rot3_part%d.o" % i) for i in range(ROT3_PARTS)]
    compiles = [base + ["-c", SRC, "-o", objs[0]]]
    compiles += [base + ["-DROT3_PART=%d" % i, "-c", ROT3_SRC, "-o", objs[1 + i]] for i in range(ROT3_PARTS)]
    objs.append(os.path.join(OBJ_DIR, "noalloc.o"))
    compiles.append(base + ["-c", NOALLOC_SRC, "-o", objs[-1]])
    compiles.append(base + ["-shared", "-o", PROBES_LIB, PROBES_SRC])
    link = [base[0], "-shared", "-o", LIB] + objs
    return compiles, link


def build(force: bool = False, verbose: bool = False) -> str:
    if (not force and os.path.exists(LIB) and os.path.exists(PROBES_LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in _deps())):
        return LIB
    import concurrent.futures as cf
    os.makedirs(OBJ_DIR, exist_ok=True)
    compiles, link = nvcc_cmds(verbose)
    with cf.ThreadPoolExecutor(len(compiles)) as pool:
        for r in pool.map(lambda c: subprocess.run(c, capture_output=True, text=True), compiles):
            if verbose or r.returncode:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode:
                raise subprocess.CalledProcessError(r.returncode, r.args)
    subprocess.run(link, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
