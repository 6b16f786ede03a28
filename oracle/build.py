"""Build the C oracle (test infrastructure) into oracle/liboracle_elph.so.

Usage: python oracle/build.py        (also called by __graft_entry__.build())
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oracle_elph.c")
LIB = os.path.join(HERE, "liboracle_elph.so")


def build(force: bool = False) -> str:
    """ORACLE_SANITIZE=1 in the environment builds with -fsanitize=address,undefined (run the CPU pins with
    LD_PRELOAD=$(gcc -print-file-name=libasan.so); see profiles/r2_sanitizers.md)."""
    san = os.environ.get("ORACLE_SANITIZE") == "1"
    if (not force and not san and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    # -O2, no -ffast-math: the oracle is meant to be plain, not tuned.
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall",
           "-o", LIB, SRC, "-lm"]
    if san:
        cmd[1:1] = ["-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
