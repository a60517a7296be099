"""Build oracle/libyee_oracle.so with gcc.  TEST INFRASTRUCTURE (see yee_oracle.c).

Flags matter: -ffp-contract=off so that no multiply-add is fused (the expression tree of
yee_oracle.c *defines* bit-exactness, SURVEY.md 8(c) reading #3); no -ffast-math; no FTZ.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libyee_oracle.so")
SRCS = [os.path.join(HERE, "yee_oracle.c"), os.path.join(HERE, "yee_oracle_impl.h")]
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-Wall"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in SRCS):
        return LIB
    cmd = ["gcc", *CFLAGS, "-o", LIB + ".tmp", SRCS[0]]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
