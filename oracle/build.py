"""Build the CPU oracle (test infrastructure) into oracle/libnh_oracle.so.

    python oracle/build.py

-O2 -ffp-contract=off keeps the FP64 arithmetic exactly as written;
-fopenmp only spreads independent cell loops over the host cores.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "nh_oracle.cpp")]
HDR = [os.path.join(HERE, "nh_oracle.h")]
# NH_ORACLE_SANITIZE=1: the same source with -fsanitize=address,undefined into a library of its own (run the
# CPU tests under it with LD_PRELOAD=$(g++ -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0)
SANITIZE = os.environ.get("NH_ORACLE_SANITIZE", "") not in ("", "0")
LIB = os.path.join(HERE, "libnh_oracle_san.so" if SANITIZE else "libnh_oracle.so")


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in SRC + HDR)


def build(force: bool = False) -> str:
    if force or stale():
        tmp = LIB + ".tmp.%d" % os.getpid()
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-Wall", "-Wextra"] + (["-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer",
                                       "-fno-sanitize-recover=undefined"] if SANITIZE else []) + ["-o", tmp] + SRC
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
