"""Build libdebye.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1306_2258_b200.build [--force]

One translation unit per group of kernel instantiations so the build parallelises; objects are cached by
mtime under csrc/build/."""
from __future__ import annotations

import concurrent.futures as cf
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(CSRC, "build")
LIB = os.path.join(HERE, "libdebye.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
# -Xfatbin=-compress-all: the device code (with its -lineinfo tables) is stored compressed, a third of the size
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
         "--expt-relaxed-constexpr", "-Xfatbin=-compress-all", *os.environ.get("DEBYE_EXTRA_NVCC_FLAGS", "").split()]


def _sources():
    return sorted(f for f in os.listdir(CSRC) if f.endswith(".cu"))


def _newest_header():
    hs = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cuh", ".h"))]
    hs.append(os.path.join(HERE, "..", "include", "debye.h"))
    return max(os.path.getmtime(h) for h in hs)


def _compile(src: str, force: bool, extra) -> str:
    obj = os.path.join(OBJ, src[:-3] + ".o")
    sp = os.path.join(CSRC, src)
    if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(sp), _newest_header()):
        subprocess.check_call([NVCC, *FLAGS, *extra, "-c", sp, "-o", obj])
    return obj


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    os.makedirs(OBJ, exist_ok=True)
    srcs = _sources()
    with cf.ThreadPoolExecutor(max_workers=min(len(srcs), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(lambda s: _compile(s, force, list(extra)), srcs))
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(o) for o in objs):
        subprocess.check_call([NVCC, "-shared", "-o", LIB, *objs, "-lcudart"])
    if verbose:
        print(LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True, extra=["-Xptxas", "-v"] if "-v" in sys.argv else [])
