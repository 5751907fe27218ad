"""Build the oracle shared library (test infrastructure; see ia_oracle.cpp header).

    python oracle/build.py              ->  oracle/libia_oracle.so
    python oracle/build.py --debug      ->  oracle/libia_oracle_debug.so  (-O1 -g, AddressSanitizer + UBSan)

The debug target is the sanitizer coverage this project can have (compute-sanitizer is closed on the GPU pool): run the
CPU suite against it with

    IA_ORACLE_DEBUG=1 LD_PRELOAD=$(g++ -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
        python -m pytest tests -q -m "not gpu"

(the sanitizer runtime has to be the first library of the process, hence the preload; leak detection is off because the
interpreter itself never frees everything).  Any report aborts the test that triggered it.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ia_oracle.cpp")
LIB = os.path.join(HERE, "libia_oracle.so")
LIB_DEBUG = os.path.join(HERE, "libia_oracle_debug.so")
COMMON = ["-std=c++17", "-fPIC", "-shared", "-fopenmp", "-frounding-math", "-ffp-contract=off",
          "-fno-fast-math", "-fno-math-errno", "-Wall", "-Wextra", "-Wno-unused-parameter"]
FLAGS = [*COMMON, "-O2"]
FLAGS_DEBUG = [*COMMON, "-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined",
               "-fno-sanitize-recover=undefined"]


def build(force: bool = False, debug: bool | None = None) -> str:
    """debug=None: the debug target iff the environment says IA_ORACLE_DEBUG=1 (how the whole suite is pointed at it)."""
    if debug is None:
        debug = os.environ.get("IA_ORACLE_DEBUG", "0") == "1"
    lib, flags = (LIB_DEBUG, FLAGS_DEBUG) if debug else (LIB, FLAGS)
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= max(os.path.getmtime(SRC), os.path.getmtime(__file__)):
        return lib
    cmd = ["g++", *flags, "-o", lib, SRC]
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, debug=True if "--debug" in sys.argv else None))
