"""Compiles the oracle's C part (oracle/nsc_oracle_sub.c) into oracle/liborc_sub.so with gcc.

    python -m oracle.build_c [--force]

TEST INFRASTRUCTURE ONLY (see oracle/nsc_oracle.py).  ``__graft_entry__.build()`` calls this so that the
checker is built next to the product; building it is not using it.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nsc_oracle_sub.c")
LIB = os.path.join(HERE, "liborc_sub.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    gcc = shutil.which("gcc")
    if gcc is None:
        raise RuntimeError("gcc not found: the oracle's C backend cannot be built")
    cmd = [gcc, "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-fcx-limited-range", SRC, "-o", LIB, "-lm"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"gcc failed:\n{r.stdout}\n{r.stderr}")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
