"""Build libpbs4d.so (the C-ABI library of include/pbs4d.h) in-tree with nvcc for sm_100a.

transport.cu is built with the default FMA contraction; grids.cu, noalloc.cu and accumulate.cu with -fmad=false (their
arithmetic must round operation by operation -- DESIGN.md "Accumulation arithmetic").
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INC = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libpbs4d.so")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", INC, "-I", CSRC]
UNITS = [("api.cu", []), ("transport.cu", []), ("grids.cu", ["-fmad=false"]), ("accumulate.cu", ["-fmad=false"]), ("roofline.cu", []),
         ("noalloc.cu", ["-fmad=false"]),
         ("delivery.cpp", []), ("tables.cpp", []), ("trials.cpp", [])]


def _sources():
    return [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INC, "pbs4d.h")]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(s) > t for s in _sources())


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    objs = []
    for src, extra in UNITS:
        obj = os.path.join(objdir, src + ".o")
        cmd = ["nvcc"] + ARCH + COMMON + extra + (["-Xptxas", "-v"] if verbose else []) + \
              ["-c", os.path.join(CSRC, src), "-o", obj]
        subprocess.run(cmd, check=True)
        objs.append(obj)
    subprocess.run(["nvcc"] + ARCH + ["-shared", "-o", LIB] + objs, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
