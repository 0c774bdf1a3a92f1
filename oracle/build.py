"""Build the oracle shared library (test infrastructure): g++ -O2 -fopenmp -shared -fPIC."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hawkes_ref.cpp")
SOURCES = [SRC, os.path.join(HERE, "tree_ref.cpp")]
# HAWKES_ORACLE_SANITIZE=1: an AddressSanitizer + UBSan build in a library of its own (run the pins under
# LD_PRELOAD=$(gcc -print-file-name=libasan.so); profiles/r02_sanitizers.md)
SANITIZE = os.environ.get("HAWKES_ORACLE_SANITIZE") == "1"
LIB = os.path.join(HERE, "libhawkes_ref_asan.so" if SANITIZE else "libhawkes_ref.so")


STAMP = LIB + ".srchash"   # sha256 of the sources the library was built from (mtimes do not survive a copy)


def _source_hash() -> str:
    import hashlib
    h = hashlib.sha256()
    for f in SOURCES:
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.exists(STAMP):
        with open(STAMP) as fh:
            if fh.read().strip() == _source_hash():
                return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra",
           "-o", tmp] + SOURCES
    if SANITIZE:
        cmd[1:1] = ["-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer", "-g"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    with open(STAMP, "w") as fh:
        fh.write(_source_hash() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force=True))
