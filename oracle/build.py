"""Build the CPU oracle (test infrastructure) into oracle/libmuca_oracle.so.

Usage: python oracle/build.py            (also called by __graft_entry__.build()
and by tests/conftest.py when the library is missing or stale).
Plain g++ -O2 with OpenMP; no CUDA, no code from the product path.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "muca_oracle.cpp")
LIB = os.path.join(HERE, "libmuca_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    # -ffp-contract=off: the fp32 acceptance (exp32, R23) is a fixed sequence of IEEE operations; no a*b+c may be fused
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB + ".tmp", SRC]
    subprocess.check_call(cmd)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
