"""Build the CPU oracle shared object (TEST INFRASTRUCTURE; see lqcd_oracle.c header).

`python oracle/build.py` or `oracle.build.build()` compiles oracle/lqcd_oracle.c twice with gcc
(fp64-input and fp32-input entry points, all arithmetic fp64) and links
oracle/liblqcd_oracle.so.  Building the checker is not using it.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lqcd_oracle.c")
LIB = os.path.join(HERE, "liblqcd_oracle.so")


def _stale() -> bool:
    return (not os.path.exists(LIB)) or os.path.getmtime(LIB) < os.path.getmtime(SRC)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    common = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-fopenmp", "-Wall", "-Wno-unknown-pragmas", "-c", SRC]
    o64 = os.path.join(HERE, "lqcd_oracle_f64in.o")
    o32 = os.path.join(HERE, "lqcd_oracle_f32in.o")
    cmds = [
        common + ["-DIN_REAL=double", "-DSUFFIX=_ref", "-DLQCD_ORACLE_FP64_BUILD", "-o", o64],
        common + ["-DIN_REAL=float", "-DSUFFIX=_ref_f32in", "-o", o32],
        ["gcc", "-shared", "-fopenmp", "-o", LIB + ".tmp", o64, o32, "-lm"],
    ]
    for c in cmds:
        if verbose:
            print(" ".join(c), file=sys.stderr)
        subprocess.run(c, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
