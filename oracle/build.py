"""Build oracle/libumi_oracle.so from oracle/umi_oracle.c with gcc.

TEST INFRASTRUCTURE, NOT PRODUCT (see umi_oracle.c).  Plain `gcc -O2 -fopenmp`,
no -ffast-math, so the arithmetic is IEEE fp64 in the order the source states.
Run as `python oracle/build.py` or call `build()`.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "umi_oracle.c")
LIB = os.path.join(HERE, "libumi_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
