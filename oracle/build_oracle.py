"""Builds oracle/libnb_oracle.so from nb_oracle.c with gcc (test infrastructure only)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nb_oracle.c")
LIB = os.path.join(HERE, "libnb_oracle.so")
FLAGS_FILE = LIB + ".flags"   # the flags the .so was built with (a box without FMA rebuilds)


def _flags() -> list[str]:
    flags = ["-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC"]
    # fmaf() as the single hardware instruction where the host has one (same correctly rounded result
    # as libm's fmaf, an order of magnitude faster in the list predicates); -ffp-contract=off still
    # forbids contracting any a*b+c that is not written as fmaf (reading A12).
    try:
        with open("/proc/cpuinfo") as fh:
            if any(line.startswith("flags") and " fma " in line + " " for line in fh):
                flags.append("-mfma")
    except OSError:
        pass
    return flags


def build(force: bool = False) -> str:
    flags = _flags()
    tag = " ".join(flags)
    built_with = None
    if os.path.exists(FLAGS_FILE):
        with open(FLAGS_FILE) as fh:
            built_with = fh.read().strip()
    if (not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC)
            and built_with == tag):
        return LIB
    subprocess.run(["gcc", *flags, "-o", LIB, SRC, "-lm"], check=True)
    with open(FLAGS_FILE, "w") as fh:
        fh.write(tag + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force=True))
