"""Build the fp64 CPU oracle (test infrastructure) into oracle/libdsk_oracle.so with plain gcc.

    python -m oracle.build

-O2, no fast-math, -ffp-contract=off (the two fp32 steps of reading O1 must stay IEEE single ops).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["orc_tree.c", "orc_moments.c", "orc_eval.c", "orc_periodic.c", "orc_bg.c", "orc_soft.c"]
LIB = os.path.join(HERE, "libdsk_oracle.so")


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + ["orc.h"])


def build(force: bool = False) -> str:
    if not force and not needs_build():
        return LIB
    cmd = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-Wall", "-Wno-unknown-pragmas", "-o", LIB] + [os.path.join(HERE, f) for f in SOURCES] + ["-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
