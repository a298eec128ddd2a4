"""Build oracle/libmlmd_ref.so from oracle/mlmd_ref.c with gcc (+OpenMP).

TEST INFRASTRUCTURE: the oracle is a checker, not part of the product path.
Called by ``__graft_entry__.build()`` and lazily by ``oracle.ref`` when the library is
missing or older than its source.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mlmd_ref.c")
LIB = os.path.join(HERE, "libmlmd_ref.so")

# -fcx-limited-range: complex products are the plain (ac-bd, ad+bc) formula, no Inf/NaN rescue
# calls.  -mavx2 -mfma: any x86-64 host of a B200 box has them; no -march=native because the
# library built on one machine travels to another.
CFLAGS = ["-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-fcx-limited-range", "-mavx2", "-mfma"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", *CFLAGS, SRC, "-o", tmp, "-lm"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
