"""Build oracle/libnb_oracle.so from oracle/nb_oracle.c with gcc (plain -O2 + OpenMP).

TEST INFRASTRUCTURE: building the checker is not using it.  Run as
`python -m oracle.build`; also called by __graft_entry__.build() and lazily
by oracle.load().
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nb_oracle.c")
LIB = os.path.join(HERE, "libnb_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared",
           "-ffp-contract=off", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
