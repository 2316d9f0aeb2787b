"""Build the CPU oracle (test infrastructure) into oracle/libchorus_oracle.so.

    python -m oracle.build

g++ -O3 -march=native -fopenmp; no CUDA and nothing taken from the CUDA package.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "chorus_oracle.cpp")
LIB = os.path.join(HERE, "libchorus_oracle.so")


LIB_SAN = os.path.join(HERE, "libchorus_oracle_san.so")


def build(force: bool = False, sanitize: bool = False) -> str:
    """sanitize: an AddressSanitizer + UndefinedBehaviorSanitizer build (tests/test_oracle_sanitizers.py runs the
    oracle's pins on it)."""
    lib = LIB_SAN if sanitize else LIB
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= os.path.getmtime(SRC)):
        return lib
    tmp = lib + f".tmp{os.getpid()}"
    opt = (["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
           if sanitize else ["-O3", "-march=native"])
    cmd = ["g++", *opt, "-fopenmp", "-std=c++17", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", tmp, SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, sanitize="--sanitize" in sys.argv))
