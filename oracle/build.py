"""Compile the fp64 CPU oracle (oracle/qxd_ref.cpp) into oracle/libqxd_ref.so with g++.

TEST INFRASTRUCTURE: building the checker is not using it.  Called by
``__graft_entry__.build()`` and lazily by ``oracle/qxd_ref.py``.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "qxd_ref.cpp")
LIB = os.path.join(HERE, "libqxd_ref.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB + ".tmp", SRC]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
