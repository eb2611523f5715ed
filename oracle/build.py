"""Builds the CPU oracle shared library (oracle/libmso.so) with gcc.

TEST INFRASTRUCTURE: called by __graft_entry__.build(), tests/ and bench.py's
cpu_baseline / --impl reference legs only.  Building the checker is not using it.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mso.c")
SRC_GRAD = os.path.join(HERE, "mso_grad.c")      # backward-pass oracle (S:Sec.8(f) NEXT-4)
LIB = os.path.join(HERE, "libmso.so")
FLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
         "-shared", "-fPIC", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    deps = [SRC, SRC_GRAD, os.path.join(HERE, "mso.h")]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.run(["gcc", *FLAGS, SRC, SRC_GRAD, "-o", tmp, "-lm"], check=True, cwd=HERE)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
