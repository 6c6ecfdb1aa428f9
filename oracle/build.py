"""Compile oracle/osog_oracle.c into oracle/libosog_oracle.so (gcc -O2 -fopenmp, no -march, no fast-math).

Called by __graft_entry__.build() and, lazily, by oracle.oracle on first import.  Building the
checker is not using it: nothing in the product path links or loads this library.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "osog_oracle.c")
LIB = os.path.join(HERE, "libosog_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-ffp-contract=off", "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
