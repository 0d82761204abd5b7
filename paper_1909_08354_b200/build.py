"""Build libsn.so in-tree (paper_1909_08354_b200/libsn.so) with nvcc for sm_100a.

The kernel translation unit is compiled once per supported line length (-DSN_LEN=N), in
parallel; nvcc cross-compiles without a GPU.  Usage: python -m paper_1909_08354_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libsn.so")
LENGTHS = (64, 128, 256, 512, 1024, 2048, 4096)   # pipelined + first-path kernels
LENGTHS_FIRST = (32,)                              # first-path kernels only
LENGTHS3 = (96, 192, 384, 768, 1536, 3072)        # 3*2^a: 12 points per thread
LENGTHS_RESIDENT = (64, 128)                       # square 2D grids held in one cluster's shared memory
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3",
         "-Xcompiler", "-fPIC", "-diag-suppress", "128"]
FLAGS += os.environ.get("SN_NVCC_EXTRA", "").split()  # tuning experiments, e.g. -DSN_CPCAP=4096


def _sources():
    out = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))]
    out.append(os.path.join(os.path.dirname(HERE), "include", "sn.h"))
    return out


def _stale(target: str) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in _sources())


def _compile(args):
    src, obj, extra = args
    if _stale(obj):
        subprocess.run([NVCC, *FLAGS, *extra, "-c", src, "-o", obj], check=True)
    return obj


def build(force: bool = False) -> str:
    """Build libsn.so if it is missing or older than its sources.  Serialised by a file lock, so several ranks of
    one node calling it at once compile once."""
    import fcntl
    os.makedirs(OBJ, exist_ok=True)
    with open(os.path.join(OBJ, ".lock"), "w") as lk:
        fcntl.flock(lk, fcntl.LOCK_EX)
        try:
            return _build_locked(force)
        finally:
            fcntl.flock(lk, fcntl.LOCK_UN)


def _build_locked(force: bool) -> str:
    if force:
        for f in os.listdir(OBJ):
            if f != ".lock":
                os.remove(os.path.join(OBJ, f))
        if os.path.exists(LIB):
            os.remove(LIB)
    if not _stale(LIB):
        return LIB
    jobs = [(os.path.join(CSRC, "sn_kernels.cu"), os.path.join(OBJ, f"sn_kernels_{n}.o"), [f"-DSN_LEN={n}"])
            for n in LENGTHS_FIRST + LENGTHS + LENGTHS3]
    jobs += [(os.path.join(CSRC, "sn_pipe.cu"), os.path.join(OBJ, f"sn_pipe_{n}.o"), [f"-DSN_LEN={n}"])
             for n in LENGTHS + LENGTHS3]
    jobs += [(os.path.join(CSRC, "sn_kernels_f64.cu"), os.path.join(OBJ, f"sn_kernels_f64_{n}.o"), [f"-DSN_LEN={n}"])
             for n in LENGTHS_FIRST + LENGTHS + LENGTHS3]     # complex128 path
    jobs += [(os.path.join(CSRC, "sn_resident.cu"), os.path.join(OBJ, f"sn_resident_{n}.o"), [f"-DSN_LEN={n}"])
             for n in LENGTHS_RESIDENT]                       # cluster-resident step of small 2D grids
    jobs.append((os.path.join(CSRC, "sn_api.cu"), os.path.join(OBJ, "sn_api.o"), []))
    jobs.append((os.path.join(CSRC, "sn_static.cu"), os.path.join(OBJ, "sn_static.o"), []))   # allocation-free entry point
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as ex:
        objs = list(ex.map(_compile, jobs))
    subprocess.run([NVCC, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a",
                    "-lcudart"], check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
