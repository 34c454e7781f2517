"""Build oracle/liblp_oracle.so from oracle/lp_oracle.c with gcc.

Flags: -O2 -ffp-contract=off (no fused multiply-add, see the header of lp_oracle.c)
and -fopenmp (the particle loops may be split over threads; arithmetic unchanged).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lp_oracle.c")
LIB = os.path.join(HERE, "liblp_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
