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
# NB_ORACLE_SANITIZE=1: an AddressSanitizer + UndefinedBehaviorSanitizer build in its own file, for running the
# pins under the sanitizers (LD_PRELOAD the gcc libasan.so into python; see profiles/r2_sanitizers.md)
SANITIZE = os.environ.get("NB_ORACLE_SANITIZE", "") not in ("", "0")
LIB = os.path.join(HERE, "libnb_oracle_asan.so" if SANITIZE else "libnb_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] \
        if SANITIZE else ["-O2"]
    cmd = ["gcc"] + opt + ["-std=c11", "-fopenmp", "-fPIC", "-shared",
                           "-ffp-contract=off", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
