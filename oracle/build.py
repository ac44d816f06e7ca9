"""Builds oracle/libcao_oracle.so from oracle/cao_oracle.cc (TEST INFRASTRUCTURE, see cao_oracle.cc)."""
from __future__ import annotations
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cao_oracle.cc")
LIB = os.path.join(HERE, "libcao_oracle.so")
# -ffp-contract=off / -fno-fast-math: every written fp32 operation is one IEEE-754 rounding.
FLAGS = ["-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", *FLAGS, SRC, "-o", tmp])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
