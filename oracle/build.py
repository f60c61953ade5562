"""Build the CPU oracle (plain C + OpenMP) into oracle/libgint_oracle.so.

Test infrastructure: building the checker is not using it.  Called by
__graft_entry__.build(), by the tests' conftest and by bench.py's cpu_baseline leg.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gint_oracle.c")
LIB = os.path.join(HERE, "libgint_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
