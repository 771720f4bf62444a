"""Build the CPU oracle (oracle/libjxo.so).  TEST INFRASTRUCTURE ONLY.

    python -m oracle.build

Plain g++, -O2, -ffp-contract=off (every add and multiply rounded separately),
no OpenMP, no -march flags: the oracle is a reference, never tuned.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "jxo.cpp")
LIB = os.path.join(HERE, "libjxo.so")
FLAGS = ["-O2", "-ffp-contract=off", "-std=c++17", "-Wall", "-Wextra", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "jxo.h")]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    cmd = ["g++", *FLAGS, "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
