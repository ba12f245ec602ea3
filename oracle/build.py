"""Build the C oracle (oracle/dd_oracle.c -> oracle/libdd_oracle.so) with gcc.  Test infrastructure only.

Run as a script (`python oracle/build.py`) or call `build()`; `__graft_entry__.build()` calls it too.
Flags are deliberately ordinary (-O2, OpenMP for the `parallel for` over DM trials); the oracle is
never tuned.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "dd_oracle.c")
LIB = os.path.join(_HERE, "libdd_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-Wall", "-Wextra",
           "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
