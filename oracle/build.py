"""Compile oracle/frost_oracle.c into oracle/libfrost_oracle.so with gcc (plain C, OpenMP).

Building the checker is not using it: __graft_entry__.build() calls this so that the tests, smoke()
and bench.py's cpu_baseline leg find the library.  -ffp-contract=off keeps every product and sum a
separately rounded IEEE operation, as the oracle's header promises.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "frost_oracle.c")
LIB = os.path.join(HERE, "libfrost_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
