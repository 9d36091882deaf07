"""Build the CPU oracle shared library (test infrastructure; see purify_oracle.cpp).

    python oracle/build.py

Plain g++ -O2 with OpenMP; no -march flags and -ffp-contract=off so that every fp32/fp64
operation is one IEEE operation (the table-index rule relies on it)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "purify_oracle.cpp")
LIB = os.path.join(HERE, "libpurify_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-fno-fast-math", SRC, "-o", LIB]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
