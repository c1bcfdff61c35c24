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
LIB_SANITIZED = os.path.join(HERE, "libtcrnet_oracle_asan.so")
# TCRNET_ORACLE_SANITIZE=1: the same sources under -fsanitize=address,undefined; the
# interpreter then has to run with LD_PRELOAD=$(gcc -print-file-name=libasan.so)
# (tests/test_oracle_pins.py::test_pins_under_address_and_ub_sanitizers does both).
SANITIZE_ENV = "TCRNET_ORACLE_SANITIZE"


def sanitizer_runtime() -> str:
    return subprocess.run(["gcc", "-print-file-name=libasan.so"], check=True, capture_output=True,
                          text=True).stdout.strip()


def build(force: bool = False) -> str:
    sanitize = os.environ.get(SANITIZE_ENV, "0") == "1"
    lib = LIB_SANITIZED if sanitize else LIB
    if not force and os.path.exists(lib) and all(os.path.getmtime(lib) >= os.path.getmtime(x) for x in SRCS):
        return lib
    tmp = lib + f".tmp{os.getpid()}"
    flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
             "-fno-omit-frame-pointer"] if sanitize else ["-O2"]
    cmd = ["gcc"] + flags + ["-std=c11", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", tmp] + SRCS
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force=True))
