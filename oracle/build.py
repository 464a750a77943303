"""Builds oracle/libnep_oracle.so from nep_oracle.c with gcc (test infrastructure only).

-ffp-contract=off: no fused multiply-adds, so the neighbour predicate
|d|^2 < r_c^2 is the plain IEEE fp64 expression the GPU side must reproduce
bit for bit (reading Q9)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nep_oracle.c")
LIB = os.path.join(HERE, "libnep_oracle.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
