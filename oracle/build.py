"""Build oracle/libdash_oracle.so from oracle/dash_oracle.c with gcc.

TEST INFRASTRUCTURE (see dash_oracle.c header).  `-ffp-contract=off` is part of the oracle's
definition: cell location is one binary32 multiply (DESIGN.md §3 Q4), never an FMA.
Run:  python oracle/build.py [--force] [--sanitize]

`--sanitize` (SURVEY.md:176) writes oracle/libdash_oracle_san.so, the same source built with
`-fsanitize=address,undefined -O1 -g`.  The pin tests run against it when DASH_ORACLE_SANITIZE=1 is set:
    LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 DASH_ORACLE_SANITIZE=1 \
        python -m pytest tests -m "not gpu" -q -k oracle
(python itself is not instrumented, so libasan must be preloaded; leak checking is off because CPython's
arenas are not freed at exit).  It is the only sanitizer tier this pool can run: compute-sanitizer is refused.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dash_oracle.c")
LIB = os.path.join(HERE, "libdash_oracle.so")
LIB_SAN = os.path.join(HERE, "libdash_oracle_san.so")


def build(force: bool = False, sanitize: bool | None = None) -> str:
    if sanitize is None:
        sanitize = os.environ.get("DASH_ORACLE_SANITIZE") == "1"
    lib = LIB_SAN if sanitize else LIB
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= os.path.getmtime(SRC)):
        return lib
    opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
           "-fno-omit-frame-pointer"] if sanitize else ["-O2"]
    cmd = ["gcc", *opt, "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-Wextra", "-shared", "-fPIC", SRC, "-o", lib + ".tmp", "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(lib + ".tmp", lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, sanitize="--sanitize" in sys.argv))
