"""Build the CPU oracle shared library (oracle/libhk_oracle.so) with gcc.

TEST INFRASTRUCTURE ONLY (see hk_oracle.c header).  Plain C, fp64, OpenMP over
bins; -ffp-contract=off so that the integer-extent formulas round exactly as
written.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hk_oracle.c")
LIB = os.path.join(HERE, "libhk_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
           "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
