"""Build the CPU oracle (test infrastructure) into oracle/libbt_oracle.so.

Flags are part of the oracle's definition: -O2, no FMA contraction, no fast-math (SURVEY 8c-R11,
R14: "the oracle is compiled with -ffp-contract=off"; the paper's own builds used fast-math,
PAPER.md l.154 -- the oracle must not).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "bt_oracle.c")
LIB = os.path.join(HERE, "libbt_oracle.so")

CFLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-fopenmp",
          "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc"] + CFLAGS + ["-o", tmp, SRC, "-lm"]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
