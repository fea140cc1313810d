"""Build the oracle shared library ``oracle/liblrmd_ref.so`` with g++.

TEST INFRASTRUCTURE (see lrmd_ref.cpp header).  Flags: -O2, no fast-math,
-ffp-contract=off so that every product and sum is individually rounded as the
source states it; OpenMP only parallelises the row index i.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lrmd_ref.cpp")
OUT = os.path.join(HERE, "liblrmd_ref.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(OUT)
            and os.path.getmtime(OUT) >= os.path.getmtime(SRC)):
        return OUT
    tmp = OUT + f".tmp{os.getpid()}"
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
           "-shared", "-fPIC", "-Wall", "-Wextra", "-o", tmp, SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, OUT)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
