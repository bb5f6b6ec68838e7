"""Build the CPU oracle (test infrastructure only) into oracle/liborc.so with gcc.

-ffp-contract=off: the accumulation oracle must round every fp32 operation once.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["orc_physics.c", "orc_transport.c", "orc_delivery.c", "orc_accumulate.c", "orc_dim.c", "orc_dvf.c", "orc_trials.c"]
LIB = os.path.join(HERE, "liborc.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, s)) > t for s in SOURCES + ["orc.h"])


def build(force: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = ["gcc", "-std=gnu11", "-O2", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-Wextra", "-o", LIB] + [os.path.join(HERE, s) for s in SOURCES] + ["-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
