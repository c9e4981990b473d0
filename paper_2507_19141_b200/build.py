"""Build paper_2507_19141_b200/libdash_hash4d.so (the C-ABI library of include/dash_hash4d.h) with nvcc
for sm_100a.  In-tree, so the .so travels to the GPU box with the repo snapshot.
Run:  python -m paper_2507_19141_b200.build [--force]
"""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdash_hash4d.so")
SOURCES = ["hash4d_kernels.cu", "bwd_runs_kernels.cu", "deform_kernels.cu", "mlp_bwd_kernels.cu", "hash4d_api.cu", "decompose_kernels.cu"]
DEPS = SOURCES + ["api_errors.h", "hash4d_kernels.h", "hash4d_plan.h", "hash4d_device.cuh", "deform_kernels.h", "deform_profile.cuh", "tcgen05_ptx.cuh", os.path.join("..", "..", "include", "dash_deform.h"), os.path.join("..", "..", "include", "dash_hash4d.h"), os.path.join("..", "..", "include", "dash_debug.h"),
               os.path.join("..", "..", "include", "dash_decompose.h")]
# The access-pattern microbenchmarks (include/dash_ceilings.h; bench.py --ceilings) are measurement tools, not the method:
# they are built into a library of their own so that the product library exports only the method.
CEIL_LIB = os.path.join(HERE, "libdash_ceilings.so")
CEIL_SOURCES = ["ceilings.cu"]
CEIL_DEPS = CEIL_SOURCES + [os.path.join("..", "..", "include", "dash_ceilings.h"),
                            os.path.join("..", "..", "include", "dash_hash4d.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-fvisibility=hidden", "-shared"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


_ID_MARK = b"DASH_BUILD_ID="
_CEIL_ID_MARK = b"DASH_CEIL_BUILD_ID="


def source_hash(deps=None) -> str:
    """sha256 over the bytes of every source and header the library is built from (mtimes do not survive rsync)."""
    h = hashlib.sha256()
    for d in sorted(DEPS if deps is None else deps):
        with open(os.path.join(CSRC, d), "rb") as fh:
            h.update(d.encode() + b"\0" + fh.read() + b"\0")
    return h.hexdigest()[:32]


def built_id(path: str = LIB, mark: bytes = _ID_MARK):
    """The source hash baked into the library (`dash_hash4d_build_id`), read from the file without loading it."""
    try:
        with open(path, "rb") as fh:
            blob = fh.read()
    except OSError:
        return None
    at = blob.find(mark)
    return None if at < 0 else blob[at + len(mark): at + len(mark) + 32].decode("ascii", "replace")


def is_stale() -> bool:
    return built_id() != source_hash()


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not is_stale():
        return LIB
    cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          [f'-DDASH_BUILD_ID_STRING="{source_hash()}"'] + \
          [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


def ceilings_is_stale() -> bool:
    return built_id(CEIL_LIB, _CEIL_ID_MARK) != source_hash(CEIL_DEPS)


def build_ceilings(force: bool = False) -> str:
    """libdash_ceilings.so: the microbenchmark kernels of include/dash_ceilings.h, nothing of the method."""
    if not force and not ceilings_is_stale():
        return CEIL_LIB
    cmd = [_nvcc()] + NVCC_FLAGS + [f'-DDASH_CEIL_BUILD_ID_STRING="{source_hash(CEIL_DEPS)}"'] + \
          [os.path.join(CSRC, s) for s in CEIL_SOURCES] + ["-o", CEIL_LIB + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(CEIL_LIB + ".tmp", CEIL_LIB)
    return CEIL_LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    print(build_ceilings(force="--force" in sys.argv))
