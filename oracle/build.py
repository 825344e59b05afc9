"""Compile oracle/nnp_oracle.c into oracle/libnnp_oracle.so (gcc, no fast-math,
no FMA contraction).  Building the checker is not using it."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nnp_oracle.c")
LIB = os.path.join(HERE, "libnnp_oracle.so")
FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c11", "-D_POSIX_C_SOURCE=200809L",
         "-shared", "-fPIC", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", *FLAGS, SRC, "-o", tmp, "-lm"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
