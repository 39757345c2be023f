"""oracle/build.py -- compile the CPU oracle's C source (TEST INFRASTRUCTURE ONLY).

gcc -O2 -fopenmp -ffp-contract=off: no fused multiply-add, so every multiply and add of the
oracle is rounded on its own (oracle section).  Building the checker is not using it:
__graft_entry__.build() calls this; nothing in the product path does.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tc_oracle.c")
LIB = os.path.join(HERE, "libtc_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-std=c11", "-Wall", "-shared", "-fPIC",
           SRC, "-o", LIB, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
