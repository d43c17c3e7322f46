"""Builds oracle/liboracle.so from oracle/hough_oracle.cpp (S1-S6) and oracle/hough_oracle_next.cpp (the NEXT rows)
(TEST INFRASTRUCTURE).

Flags: -O2, no FMA contraction, no fast-math, so that every fp32 operation in
the oracle rounds once, as written (reading Q12).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hough_oracle.cpp")
SRCS = [SRC, os.path.join(HERE, "hough_oracle_next.cpp")]
LIB = os.path.join(HERE, "liboracle.so")
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", "-pthread"]


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in SRCS):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["g++", *FLAGS, "-o", tmp, *SRCS])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
