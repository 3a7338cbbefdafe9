"""Build liboracle (oracle/axo_oracle.cpp) with g++.  Test infrastructure only.

    python -m oracle.build          # builds oracle/libaxo_oracle.so if stale
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "axo_oracle.cpp")
LIB = os.path.join(HERE, "libaxo_oracle.so")
# -ffp-contract=off: the only fused operation is the explicit fmaf of O1 (reading A-22)
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fvisibility=hidden", "-shared", "-fPIC", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["g++", *FLAGS, SRC, "-o", tmp]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
