"""Compile oracle/sw_oracle.cpp into oracle/libsw_oracle.so with g++ (no CUDA).

Usage: python -m oracle.build     (also called by __graft_entry__.build())
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sw_oracle.cpp")
HDR = os.path.join(HERE, "sw_oracle.h")
SRC_XY = os.path.join(HERE, "sw_xy_oracle.cpp")     # the XY extension: same library
HDR_XY = os.path.join(HERE, "sw_xy_oracle.h")
LIB = os.path.join(HERE, "libsw_oracle.so")


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(f) for f in (SRC, HDR, SRC_XY, HDR_XY))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    # -ffp-contract=off: the XY oracle spells out every fused multiply-add itself (sw_xy_oracle.h, "Arithmetic")
    cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra", "-ffp-contract=off",
           "-fvisibility=default", "-o", LIB, SRC, SRC_XY]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
