"""Builds the C-ABI library ``libbie_b200.so`` in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2108_01786_b200.build [--force] [--clean] [--verbose]

The library exports the calls declared in ``include/bie.h``.  It links the CUDA runtime statically, so it
loads on a machine without a driver (every call then fails with BIE_ERR_DEVICE) and does not depend on
which libcudart PyTorch ships.  Every ``csrc/*.cu`` is compiled to its own object under ``build/`` (git-ignored), the
files in parallel, and only the objects older than their source, a header, this file or the flags are rebuilt
(``--force`` links again whatever the dates say, e.g. after changing BIE_NVCC_EXTRA; ``--clean`` drops the objects first).
"""
from __future__ import annotations

import concurrent.futures
import glob
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libbie_b200.so")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--fmad=true",            # default; no fast-math anywhere: FP64 arithmetic is IEEE except bie_rcp()
    "-Xcompiler", "-fPIC",
]
LINK_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(INCLUDE, "*.h")) + [__file__]


def _extra():
    return os.environ.get("BIE_NVCC_EXTRA", "").split()   # e.g. -DBIE_PHASE_TIMING (developer builds only)


def _obj(src: str) -> str:
    tag = hashlib.sha1(" ".join(NVCC_FLAGS + _extra()).encode()).hexdigest()[:10]
    return os.path.join(OBJ, os.path.splitext(os.path.basename(src))[0] + "." + tag + ".o")


def _obj_stale(src: str) -> bool:
    o = _obj(src)
    if not os.path.exists(o):
        return True
    t = os.path.getmtime(o)
    return any(os.path.getmtime(d) > t for d in [src] + _headers())


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)     # the objects need not exist (they do not travel to the GPU box): the library is judged by its sources
    return any(os.path.getmtime(d) > t for d in sources() + _headers())


def _compile(nvcc: str, src: str, verbose: bool) -> None:
    tmp = _obj(src) + f".{os.getpid()}.tmp"
    cmd = [nvcc] + NVCC_FLAGS + _extra() + (["-Xptxas", "-v"] if verbose else []) + ["-I", INCLUDE, "-c", "-o", tmp, src]
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    subprocess.check_call(cmd)
    os.replace(tmp, _obj(src))


def build_library(force: bool = False, verbose: bool = False, clean: bool = False) -> str:
    if not force and not clean and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    if clean:
        for o in glob.glob(os.path.join(OBJ, "*.o")):
            os.remove(o)
    todo = [s for s in sources() if _obj_stale(s)]
    with concurrent.futures.ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as ex:
        for f in [ex.submit(_compile, nvcc, s, verbose) for s in todo]:
            f.result()
    tmp = LIB + f".{os.getpid()}.tmp"
    subprocess.check_call([nvcc] + LINK_FLAGS + ["-o", tmp] + [_obj(s) for s in sources()])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build_library(force="--force" in sys.argv, verbose="--verbose" in sys.argv, clean="--clean" in sys.argv))
