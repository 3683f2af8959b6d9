"""Compile the CPU oracle (test infrastructure) into oracle/liborc.so with gcc.

Usage: python -m oracle.build
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sph_oracle.c")
LIB = os.path.join(HERE, "liborc.so")

# -ffp-contract=off: the canonical conversions (C1) and the fp32 predicate (C2) need
# individually rounded IEEE operations.  No -ffast-math, no -march=native.
CMD = ["gcc", "-std=c11", "-O2", "-fopenmp", "-ffp-contract=off", "-fvisibility=hidden",
       "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = list(CMD)
    cmd[cmd.index(LIB)] = tmp
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
