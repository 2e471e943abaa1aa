"""Compile the CPU oracle (plain C, gcc, OpenMP) into oracle/libdtn_oracle.so.
Building the checker is not using it: __graft_entry__.build() calls this.

Sanitizer mode: with ORACLE_SANITIZE=1 in the environment the oracle is built with
-fsanitize=address,undefined into oracle/libdtn_oracle_san.so and that library is the one loaded; run the CPU pins
under it with

    LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)" ASAN_OPTIONS=detect_leaks=0 \
    ORACLE_SANITIZE=1 python -m pytest tests -q -m "not gpu" -k oracle
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dtn_oracle.c")
LIB = os.path.join(HERE, "libdtn_oracle.so")
LIB_SAN = os.path.join(HERE, "libdtn_oracle_san.so")


def build(force: bool = False) -> str:
    sanitize = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
    lib = LIB_SAN if sanitize else LIB
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(SRC):
        return lib
    flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if sanitize else ["-O2"]
    cmd = ["gcc", *flags, "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-Wall", "-Wextra", "-o", lib, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    print(build(force=True))
