"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, not product code).

    python oracle/build.py            # -> oracle/libgeo_oracle.so

Flags: -O2 -ffp-contract=off (no FMA contraction: plain IEEE arithmetic in the
written order).  Called by __graft_entry__.build() and by oracle/geo_oracle.py
on first use.  Building the checker is not using it.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "geo_oracle.cpp")
SRCS = [SRC, os.path.join(HERE, "geo_tab_oracle.cpp")]      # fixed-step/adaptive analytic metrics; tabulated metrics (8(f).3)
LIB = os.path.join(HERE, "libgeo_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(x) for x in SRCS):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
           "-Wall", "-Wextra", "-o", LIB + ".tmp"] + SRCS
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
