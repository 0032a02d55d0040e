"""Builds oracle/libkvr_oracle.so from oracle/kvr_oracle.c and oracle/kvr_attention_oracle.c with gcc.

ORACLE = test infrastructure (see the header of kvr_oracle.c).  Building the
checker is not using it: __graft_entry__.build() calls build() here; only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs load the result.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, f) for f in ("kvr_oracle.c", "kvr_attention_oracle.c")]
LIB = os.path.join(HERE, "libkvr_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in SRCS)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-Wextra", "-shared", "-fPIC", *SRCS, "-o", LIB + ".tmp", "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
