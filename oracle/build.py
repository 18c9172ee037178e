"""Build the fp64 CPU oracle (oracle/asm_oracle.c) into oracle/liboracle_asm.so with gcc.

Test infrastructure only (see the header of asm_oracle.c).  Called by oracle/asm_oracle.py on
first use and by __graft_entry__.build(); building the checker is not using it.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "asm_oracle.c")
LIB = os.path.join(HERE, "liboracle_asm.so")


def build(force: bool = False) -> str:
    """Compile if the .so is missing or older than the source; return its path."""
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-shared", "-fPIC", "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
