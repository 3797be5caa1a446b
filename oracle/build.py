"""Build the CPU oracle (oracle/vro.c -> oracle/libvro.so).  TEST INFRASTRUCTURE.

gcc, double precision, no FMA contraction (so results do not depend on the host's ISA),
OpenMP over pixels.  Called by __graft_entry__.build() and, lazily, by oracle/vro.py.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "vro.c")
HDR = os.path.join(HERE, "vro.h")
LIB = os.path.join(HERE, "libvro.so")


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = ["gcc", "-std=gnu11", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
