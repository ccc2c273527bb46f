"""Builds oracle/libgs_oracle.so from oracle/gs_oracle.cpp with g++ (no CUDA, no product code)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libgs_oracle.so")
SRC = [os.path.join(HERE, "gs_oracle.cpp")]
DEPS = SRC + [os.path.join(HERE, "gs_oracle.h")]
# -ffp-contract=off: no FMA contraction, so every fp32 operation of C-P0..C-P8 rounds once.
FLAGS = ["-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math", "-pthread", "-Wall"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    cmd = ["g++"] + FLAGS + ["-o", LIB] + SRC
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
