"""Build the oracle shared library (test infrastructure; see ia_oracle.cpp header).

    python oracle/build.py        ->  oracle/libia_oracle.so
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ia_oracle.cpp")
LIB = os.path.join(HERE, "libia_oracle.so")
FLAGS = ["-std=c++17", "-O2", "-fPIC", "-shared", "-fopenmp", "-frounding-math", "-ffp-contract=off",
         "-fno-fast-math", "-fno-math-errno", "-Wall", "-Wextra", "-Wno-unused-parameter"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", *FLAGS, "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
