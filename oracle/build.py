"""Build oracle/libdash_oracle.so from oracle/dash_oracle.c with gcc.

TEST INFRASTRUCTURE (see dash_oracle.c header).  `-ffp-contract=off` is part of the oracle's
definition: cell location is one binary32 multiply (DESIGN.md §3 Q4), never an FMA.
Run:  python oracle/build.py
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dash_oracle.c")
LIB = os.path.join(HERE, "libdash_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-Wextra", "-shared", "-fPIC", SRC, "-o", LIB + ".tmp", "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
