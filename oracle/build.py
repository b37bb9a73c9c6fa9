"""Build the ORACLE shared library (test infrastructure, not the product).

    python oracle/build.py

g++ -O2 -ffp-contract=off (no FMA contraction, no fast-math) so the oracle's
arithmetic is exactly the operation sequence written in ark_oracle.cpp.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ark_oracle.cpp")
LIB = os.path.join(HERE, "libark_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math",
           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
