"""Count the FP64 instructions of one RK4 step in the compiled kernel (static SASS count).

    python -m paper_1803_08320_b200.sass_count [kernel-substring]

Finds the innermost hot loop of a geo_rk4_kernel instantiation in libgeo.so (the backward branch that
spans the most DFMA) and prints DFMA / DMUL / DADD / DSETP / MUFU / total instruction counts inside it,
and flop = 2*DFMA + DMUL + DADD.  bench.py's FLOP_PER_STEP constants and DESIGN.md's "algorithmic work
per unit" come from this count (cold paths that sit inside the loop's address range but run once per
particle are excluded by counting only up to the first cold-path call, see --raw to disable).
"""
from __future__ import annotations

import re
import subprocess
import sys

from . import build

_INS = re.compile(r"^\s+/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)(.*?);")


def kernels() -> dict:
    out = subprocess.run(["cuobjdump", "-sass", build.build()], capture_output=True, text=True, check=True).stdout
    res, name = {}, None
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            name = m.group(1)
            res[name] = []
            continue
        m = _INS.match(line)
        if m and name:
            res[name].append((int(m.group(1), 16), m.group(2), m.group(3)))
    return res


def hot_loop(ins: list) -> tuple[int, int]:
    """Address range [lo, hi] of the backward branch enclosing the most DFMA."""
    best = (0, 0, -1)
    for addr, op, rest in ins:
        if op.startswith("BRA"):
            m = re.search(r"0x([0-9a-f]+)", rest)
            if m:
                tgt = int(m.group(1), 16)
                if tgt < addr:
                    n = sum(1 for a, o, _ in ins if tgt <= a <= addr and o.startswith("DFMA"))
                    if n > best[2]:
                        best = (tgt, addr, n)
    return best[0], best[1]


def count(name_part: str = "ILb1ELi0ELb0") -> dict:
    ks = kernels()
    name = next(k for k in ks if "_kernel" in k and name_part in k)
    ins = ks[name]
    lo, hi = hot_loop(ins)
    body = [(a, o) for a, o, _ in ins if lo <= a <= hi]
    c = {"kernel": name, "loop": (hex(lo), hex(hi)), "total": len(body)}
    for key in ("DFMA", "DMUL", "DADD", "DSETP", "MUFU"):
        c[key] = sum(1 for _, o in body if o.startswith(key))
    c["fp64_pipe"] = c["DFMA"] + c["DMUL"] + c["DADD"] + c["DSETP"]
    c["flop"] = 2 * c["DFMA"] + c["DMUL"] + c["DADD"]
    return c


if __name__ == "__main__":
    part = sys.argv[1] if len(sys.argv) > 1 else "ILb1ELi0ELb0"
    for k, v in count(part).items():
        print(f"{k}: {v}")
