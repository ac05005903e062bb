"""Compile the fp64 oracle (oracle/sopo.c) into oracle/libsopo.so with gcc.  Test infrastructure only."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sopo.c")
LIB = os.path.join(HERE, "libsopo.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "sopo.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
           SRC, "-o", LIB, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
