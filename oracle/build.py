"""Compile oracle/tcrnet_oracle.c + oracle/network_oracle.c into oracle/libtcrnet_oracle.so with gcc.

TEST INFRASTRUCTURE.  Building the checker is not using it: __graft_entry__.build()
calls this; only tests/, smoke() and bench.py's cpu_baseline / --impl reference legs
load the result.  -O2, no tuning flags: the oracle is never optimised.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "tcrnet_oracle.c"), os.path.join(HERE, "network_oracle.c")]
LIB = os.path.join(HERE, "libtcrnet_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(x) for x in SRCS):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", tmp] + SRCS
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
