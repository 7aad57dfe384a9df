"""Build the CPU oracle (oracle/xy_oracle.c) into oracle/libxy_oracle.so.

TEST INFRASTRUCTURE: only tests/, __graft_entry__ (build/smoke) and bench.py's
cpu_baseline / --impl reference legs may call this.  Flags matter:
-ffp-contract=off keeps every fp64 operation a single IEEE operation in the
order written (the oracle's arithmetic is specified to the rounding).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "xy_oracle.c")
LIB = os.path.join(HERE, "libxy_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-Wextra", "-shared", "-fPIC", SRC, "-o", LIB, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
