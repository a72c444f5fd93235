"""Compile oracle/ts_oracle.c into oracle/libts_oracle.so (TEST INFRASTRUCTURE ONLY).

Flags per SURVEY.md section 8(c) O8: no fast-math, no FMA contraction.
Usage: python -m oracle.build
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ts_oracle.c")
LIB = os.path.join(HERE, "libts_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm", "-lpthread"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
