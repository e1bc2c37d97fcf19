"""In-tree build of liblh.so for sm_100a (nvcc cross-compiles without a GPU)."""
from __future__ import annotations

import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblh.so")
SOURCES = ["lh_api.cu", "lh_kernels.cu", "lh_delens.cu", "lh_noalloc.cu", "lh_pack.cpp"]
HEADERS = ["lh_kernels.h", "lh_pack.h", "lh_math.cuh", os.path.join("..", "..", "include", "lh.h"),
           os.path.join("..", "..", "include", "lh_diag.h")]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared",
]


def source_hash() -> str:
    """SHA-256 over the sources and headers, in list order; compiled into the library as lh_source_hash()."""
    h = hashlib.sha256()
    for f in SOURCES + HEADERS:
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def _hash_flag() -> str:
    return f'-DLH_SOURCE_HASH="{source_hash()}"'


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


LIB_CHECK = os.path.join(HERE, "liblh_check.so")


def build_check(force: bool = False) -> str:
    """The CHECKING build of the same sources (-DLH_BOUNDS_CHECK): every global-memory access of the superposition kernel
    is compared with the address ranges the launch was given; a stand-in for compute-sanitizer memcheck, which is
    closed on this GPU pool.  Test infrastructure (tests/test_gpu_bounds.py); never loaded by the product path."""
    stale = not os.path.exists(LIB_CHECK) or any(
        os.path.getmtime(os.path.join(CSRC, f)) > os.path.getmtime(LIB_CHECK) for f in SOURCES + HEADERS)
    if force or stale:
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc, *NVCC_FLAGS, _hash_flag(), "-DLH_BOUNDS_CHECK", "-o", LIB_CHECK] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB_CHECK


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "nvcc")
        cmd = [nvcc, *NVCC_FLAGS, _hash_flag(), "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.run(cmd, check=True, cwd=CSRC)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
