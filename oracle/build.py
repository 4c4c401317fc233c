"""Build the CPU oracle (oracle/ts_oracle.c) into oracle/libts_oracle.so with gcc.

TEST INFRASTRUCTURE ONLY -- see the header of ts_oracle.c.  No -ffast-math (reading A13).
Run as `python oracle/build.py`, or call `build()`; `__graft_entry__.build()` calls it too.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ts_oracle.c")
LIB = os.path.join(HERE, "libts_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
