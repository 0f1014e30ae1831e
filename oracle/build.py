"""Build the CPU oracle (TEST INFRASTRUCTURE) into oracle/liboracle.so.

Flags follow DESIGN.md: -O2 -ffp-contract=off, no -ffast-math, so that every formula is
evaluated exactly as typed in gst_oracle.hpp.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "oracle_capi.cpp")]
HDR = [os.path.join(HERE, "gst_oracle.hpp")]
OUT = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in SRC + HDR)
    if not force and os.path.exists(OUT) and os.path.getmtime(OUT) >= newest:
        return OUT
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
           "-Wall", "-o", OUT] + SRC + ["-lquadmath"]
    subprocess.check_call(cmd, cwd=HERE)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
