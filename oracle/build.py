"""Build the oracle shared library (oracle/libfaro.so) with g++.  Test infrastructure only.

-ffp-contract=off: every FP64 operation in faro.cpp is one rounded IEEE operation (no FMA),
which is what the bit-exactness definitions in DESIGN.md rely on.  No -march flag: the
library built here also runs on the GPU box's host CPU.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "faro.cpp")
OUT = os.path.join(HERE, "libfaro.so")


def build(force=False):
    deps = [SRC, os.path.join(HERE, "faro.h")]
    if not force and os.path.exists(OUT) and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps):
        return OUT
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", OUT, SRC]
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
