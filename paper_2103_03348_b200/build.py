"""In-tree build of the CUDA library (sm_100a only):  python -m paper_2103_03348_b200.build"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhawkes_b200.so")
LIB_GUARD = os.path.join(HERE, "libhawkes_b200_guard.so")   # debug build: -DHAWKES_GUARD (hawkes_debug_guard_check)
SOURCES = [os.path.join(CSRC, "hawkes.cu"), os.path.join(CSRC, "tree.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("exp2_consts.inc", "pass1_sym.cuh", "hmc_kmat.cuh", "hmc_ksparse.cuh", "skip.cuh", "cross.cuh", "shard.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "hawkes.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v", "--expt-relaxed-constexpr"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


STAMP = LIB + ".srchash"   # sha256 of the sources the library was built from (mtimes do not survive a copy of the tree)


def source_hash() -> str:
    import hashlib
    h = hashlib.sha256()
    for d in DEPS:
        h.update(os.path.basename(d).encode())
        with open(d, "rb") as fh:
            h.update(fh.read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()


def up_to_date(guard: bool = False) -> bool:
    lib = LIB_GUARD if guard else LIB
    if not (os.path.exists(lib) and os.path.exists(lib + ".srchash")):
        return False
    with open(lib + ".srchash") as fh:
        return fh.read().strip() == source_hash()


def build(force: bool = False, verbose: bool = False, guard: bool = False) -> str:
    lib = LIB_GUARD if guard else LIB
    if not force and up_to_date(guard):
        return lib
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [nvcc()] + NVCC_FLAGS + (["-DHAWKES_GUARD"] if guard else []) + ["-o", tmp] + SOURCES
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    if not guard:
        with open(os.path.join(HERE, "ptxas_info.log"), "w") as fh:
            fh.write(res.stderr)
    os.replace(tmp, lib)
    with open(lib + ".srchash", "w") as fh:
        fh.write(source_hash() + "\n")
    return lib


if __name__ == "__main__":
    print(build(force=True, verbose="-v" in sys.argv, guard="--guard" in sys.argv))
