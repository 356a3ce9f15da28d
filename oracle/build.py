"""ORACLE — TEST INFRASTRUCTURE ONLY.  Builds oracle/libmfo.so with g++ (no CUDA, no GPU).

    python oracle/build.py

Flags: -O2 -ffp-contract=off (no fused multiply-add: every rounding is the one written in the source).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libmfo.so")
SOURCES = ["mfo.cpp"]
HEADERS = ["mfo.h", "real.hpp", "method.hpp", "amplitude.hpp", "amplitude_qq.hpp"]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + HEADERS)


def build(force=False):
    if not force and not needs_build():
        return LIB
    cmd = ["g++", "-std=gnu++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wno-unused",
           "-o", LIB] + [os.path.join(HERE, s) for s in SOURCES] + ["-lquadmath"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
