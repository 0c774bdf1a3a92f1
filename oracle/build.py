"""Build the oracle shared library (test infrastructure): g++ -O2 -fopenmp -shared -fPIC."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hawkes_ref.cpp")
SOURCES = [SRC, os.path.join(HERE, "tree_ref.cpp")]
LIB = os.path.join(HERE, "libhawkes_ref.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(f) for f in SOURCES)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra",
           "-o", tmp] + SOURCES
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
