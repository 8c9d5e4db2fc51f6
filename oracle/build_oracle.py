"""Compile the fp64 CPU oracle (test infrastructure) into oracle/libwstack_oracle.so.

-ffp-contract=off: the position rule is a fixed sequence of correctly rounded binary64
operations with explicit fma(); no -march flags, so the library runs on any x86-64 host
(glibc's fma() picks the hardware instruction at run time).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "wstack_oracle.c")
LIB = os.path.join(HERE, "libwstack_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
