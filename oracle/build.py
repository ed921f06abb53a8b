"""Build the CPU oracle shared library (TEST INFRASTRUCTURE, not product code).

    python oracle/build.py            # -> oracle/libgeo_oracle.so

Flags: -O2 -ffp-contract=off (no FMA contraction: plain IEEE arithmetic in the
written order).  Called by __graft_entry__.build() and by oracle/geo_oracle.py
on first use.  Building the checker is not using it.

    python oracle/build.py --sanitize # -> oracle/libgeo_oracle_san.so

the same sources under -fsanitize=address,undefined (tests/test_oracle_sanitizers.py
loads it in a child process with GEO_ORACLE_SANITIZE=1 and libasan preloaded).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "geo_oracle.cpp")
SRCS = [SRC, os.path.join(HERE, "geo_tab_oracle.cpp"),     # fixed-step/adaptive analytic metrics; tabulated metrics (8(f).3)
        os.path.join(HERE, "geo_ks_oracle.cpp")]            # Kerr in Cartesian Kerr-Schild coordinates (8(f).3, second clause)
LIB = os.path.join(HERE, "libgeo_oracle.so")
LIB_SAN = os.path.join(HERE, "libgeo_oracle_san.so")


def build(force: bool = False, sanitize: bool | None = None) -> str:
    """sanitize=None: follow the environment (GEO_ORACLE_SANITIZE=1 selects the ASan/UBSan build)."""
    if sanitize is None:
        sanitize = os.environ.get("GEO_ORACLE_SANITIZE") == "1"
    lib = LIB_SAN if sanitize else LIB
    deps = SRCS + [os.path.join(HERE, "dp45.h")]
    if not force and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(x) for x in deps):
        return lib
    opt = (["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
           if sanitize else ["-O2"])
    tmp = f"{lib}.tmp{os.getpid()}"
    cmd = ["g++"] + opt + ["-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
                           "-Wall", "-Wextra", "-o", tmp] + SRCS
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    return lib


def sanitizer_runtime() -> str:
    """Path of libasan.so to LD_PRELOAD into a python process that loads the sanitized oracle."""
    return subprocess.run(["g++", "-print-file-name=libasan.so"], capture_output=True, text=True, check=True).stdout.strip()


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, sanitize=True if "--sanitize" in sys.argv else None))
