"""Build oracle/liboracle.so from staggered_oracle.c with gcc (test infrastructure only)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "staggered_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")

CMD = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
       "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        subprocess.run(CMD, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
