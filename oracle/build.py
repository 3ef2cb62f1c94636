"""Build liboracle.so (plain C, gcc).  TEST INFRASTRUCTURE: the CUDA path never calls this."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "bz_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")
CFLAGS = ["-O2", "-std=c11", "-Wall", "-ffp-contract=off", "-mfma", "-fopenmp", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "bz_oracle.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    subprocess.check_call(["gcc", *CFLAGS, "-o", LIB, SRC, "-lm"])
    return LIB


if __name__ == "__main__":
    print(build(force=True))
