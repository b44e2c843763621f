"""Build oracle/libmlp_oracle.so from oracle/mlp_oracle.c with gcc (test infrastructure only).

Usage: python oracle/build.py     (also called by __graft_entry__.build()).
-ffp-contract=off keeps gcc from fusing a*b+c into an fma, so every product and sum in the
oracle is rounded exactly as written.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mlp_oracle.c")
LIB = os.path.join(HERE, "libmlp_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-fno-fast-math", "-ffp-contract=off", "-fopenmp", "-std=c99",
           "-Wall", "-Wextra", "-shared", "-fPIC", "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
