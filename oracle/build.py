"""Build the CPU oracle shared library (TEST INFRASTRUCTURE ONLY).

g++ -O2 -ffp-contract=off, never -ffast-math: the quantiser's fp32 steps must be plain IEEE
(reading #8).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "grinqh_oracle.cpp")
LIB = os.path.join(HERE, "libgrinqh_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
