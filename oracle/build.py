"""Compile oracle/bfly_oracle.c into oracle/libbfly_oracle.<cpu>.so with gcc.

TEST INFRASTRUCTURE.  Flags: -O2 -fopenmp -ffp-contract=off (no -ffast-math), so that
every float64 sum is evaluated in the order the source states.  The library name
carries a hash of the host's CPU flags because it is built with -march=native and
the repository snapshot (built .so included) travels between machines.
"""
from __future__ import annotations

import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "bfly_oracle.c")


def _cpu_tag() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags"):
                    flags = line
                    break
    except OSError:
        pass
    return hashlib.sha1(flags.encode()).hexdigest()[:10]


LIB = os.path.join(HERE, f"libbfly_oracle.{_cpu_tag()}.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O2", "-ftree-vectorize", "-march=native", "-fopenmp",
           "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", "-std=c11",
           SRC, "-o", tmp, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
