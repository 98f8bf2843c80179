"""Builds the CPU oracle (oracle/libqtam_ref.so) with g++.  Test infrastructure only.

-ffp-contract=off keeps the binary32 threshold variant free of fused multiply-adds (see
qtam_ref_threshold_rowmedian_f32); -O2 without -ffast-math keeps IEEE semantics everywhere.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "qtam_ref.cpp")
HDR = os.path.join(HERE, "qtam_ref.h")
LIB = os.path.join(HERE, "libqtam_ref.so")


def build(force: bool = False) -> str:
    stale = force or not os.path.exists(LIB) or any(
        os.path.getmtime(s) > os.path.getmtime(LIB) for s in (SRC, HDR))
    if stale:
        cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-Wall", "-Wextra", "-o", LIB, SRC]
        subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
