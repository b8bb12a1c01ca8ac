"""Build step for the CPU oracle (test infrastructure): g++ -> oracle/liboracle.so.

Run as `python -m oracle.build` or call `build()`.  The flags are part of the oracle's contract:
`-ffp-contract=off` keeps every `a*b+c` as two roundings (the explicit `fmaf` calls stay fused);
`-mfma` is added when the host CPU has FMA so `fmaf` inlines to one instruction (same value either
way, glibc's software fmaf is exact too -- only slower).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mi_oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")


def _cpu_has(flag: str) -> bool:
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    return flag in line.split()
    except OSError:
        pass
    return False


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC"]
    if _cpu_has("fma"):
        cmd.append("-mfma")
    if _cpu_has("sse4_1"):
        cmd.append("-msse4.1")  # inline floorf
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd += ["-o", tmp, SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
