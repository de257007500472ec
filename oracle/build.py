"""Compile the CPU oracle (oracle/gf_oracle.c) into oracle/libgf_oracle.so.

TEST INFRASTRUCTURE: building the checker is not using it.  Called by
``__graft_entry__.build()`` and, lazily, by ``oracle.load()``.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gf_oracle.c")
LIB = os.path.join(HERE, "libgf_oracle.so")

# -ffp-contract=off: no FMA contraction, so the oracle's rounding does not depend on the
# host's ISA.  -fcx-limited-range: complex products are the textbook (ac-bd) + i(ad+bc).
CFLAGS = ["-O2", "-std=c99", "-ffp-contract=off", "-fcx-limited-range", "-fopenmp",
          "-shared", "-fPIC", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", *CFLAGS, SRC, "-o", LIB, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
