"""Compile synth/fps.c (farthest-point sampling of the candidate points, an input generator) into
synth/libsynth_fps.so with gcc.  `__graft_entry__.build()` calls this; `fps_samples` builds
it on first use when it is missing."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "fps.c")
LIB = os.path.join(HERE, "libsynth_fps.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O3", "-std=c99", "-fPIC", "-shared", "-ffp-contract=off", "-ffinite-math-only", "-fno-signed-zeros", "-Wall", "-Wextra",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
