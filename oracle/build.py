"""Compile the CPU oracle (oracle/lpc_oracle.c) into oracle/liblpc_oracle.so.

TEST INFRASTRUCTURE: building the checker is not using it.  Called by
``__graft_entry__.build()`` and, lazily, by ``oracle/lpc_oracle.py``.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lpc_oracle.c")
LIB = os.path.join(HERE, "liblpc_oracle.so")

CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, SRC, "-lm"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
