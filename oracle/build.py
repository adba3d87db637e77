"""Build the CPU oracle (TEST INFRASTRUCTURE ONLY) into oracle/libpat_oracle.so.

The flags are part of the oracle's definition: -ffp-contract=off keeps
u = tau*fs a single IEEE fp32 multiply (reading R8); no -ffast-math,
no -march=native.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pat_oracle.c")
LIB = os.path.join(HERE, "libpat_oracle.so")
FLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.run(["gcc", *FLAGS, "-o", tmp, SRC, "-lm"], check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
