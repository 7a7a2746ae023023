"""Build the CPU fp64 oracle (oracle/blip_oracle.c) into oracle/libblip_oracle.so with gcc.

TEST INFRASTRUCTURE ONLY (see oracle/blip_oracle.c header).  `-ffp-contract=off` pins the
IEEE sequence of the cell-index map; `-O2`, no fast-math.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "blip_oracle.c")
LIB = os.path.join(HERE, "libblip_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC",
           "-shared", "-std=c11", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
