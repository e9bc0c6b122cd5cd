"""Build oracle/libfd_oracle.so from oracle/fd_oracle.c (TEST INFRASTRUCTURE, not product code).

gcc -O2 -fopenmp, no -ffast-math: the oracle is the plain definition (oracle/fd_oracle.c header).
Run `python -m oracle.build` or call build(); tests and __graft_entry__.build() do the latter.
"""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "fd_oracle.c")
LIB = os.path.join(_HERE, "libfd_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
