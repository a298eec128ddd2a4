"""Build the C-ABI CUDA library in-tree with nvcc for sm_100a.

    libmlmd.so       the product: every csrc/*.cu except the test hooks; hidden visibility, so it exports
                     exactly the functions include/mlmd.h declares
    libmlmd_test.so  the same objects plus csrc/test_hooks.cu (kernel-level entry points that tests/ call
                     to check single GEMM kernels against dense products); never loaded by the product
"""
from __future__ import annotations

import glob
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libmlmd.so")
TEST_LIB = os.path.join(HERE, "libmlmd_test.so")
TEST_ONLY = {"test_hooks.cu"}
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

COMPILE_FLAGS = [
    "-O3", "-std=c++17", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden",
]
LINK_FLAGS = ["-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _headers():
    return glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(HERE, "..", "include", "*.h"))


def _stale(target, deps):
    return not os.path.exists(target) or any(os.path.getmtime(target) < os.path.getmtime(f) for f in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    srcs, hdrs = sources(), _headers()
    if not force and not _stale(LIB, srcs + hdrs) and not _stale(TEST_LIB, srcs + hdrs):
        return LIB
    os.makedirs(OBJ, exist_ok=True)

    def compile_one(src):
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
        if force or _stale(obj, [src] + hdrs):
            subprocess.check_call([NVCC, *COMPILE_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-c", src, "-o", obj])
        return obj

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
        objs = list(ex.map(compile_one, srcs))
    product = [o for o, s in zip(objs, srcs) if os.path.basename(s) not in TEST_ONLY]
    for lib, members in ((LIB, product), (TEST_LIB, objs)):
        tmp = lib + ".tmp.%d" % os.getpid()
        subprocess.check_call([NVCC, *LINK_FLAGS, *members, "-o", tmp])
        os.replace(tmp, lib)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
