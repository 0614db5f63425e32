"""Compile the fp64 CPU oracle (oracle/gsvox_oracle.c) into oracle/libgsvox_oracle.so.

TEST INFRASTRUCTURE ONLY — see the header of gsvox_oracle.c.  Building the checker
is not using it: __graft_entry__.build() calls this, the product never does.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gsvox_oracle.c")
LIB = os.path.join(HERE, "libgsvox_oracle.so")

# -ffp-contract=off: one IEEE rounding per fp64 operation (box bounds, reading A5).
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
          "-std=c11", "-Wall", "-Wextra", "-Wno-unused-variable"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.run(["gcc", *CFLAGS, "-o", tmp, SRC, "-lm"], check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
