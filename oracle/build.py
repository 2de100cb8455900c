"""Build the CPU oracle (test infrastructure) into oracle/libsldg_oracle.so with gcc.

-ffp-contract=off: the oracle's arithmetic is exactly the C expressions written in
sldg_oracle.c (no fused multiply-add), so integer decisions such as s = floor(delta)
are taken in plain fp64 ("same precision" rule).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sldg_oracle.c")
LIB = os.path.join(HERE, "libsldg_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
