"""Build the CPU oracle (plain C, gcc) into oracle/liboracle_dd4dvar.so.

Test infrastructure only: see the header of dd4dvar_oracle.c.  -ffp-contract=off keeps every
multiply and add separately rounded, as written.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dd4dvar_oracle.c")
LIB = os.path.join(HERE, "liboracle_dd4dvar.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=gnu99", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-Wno-unused-variable", "-Wno-maybe-uninitialized", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
