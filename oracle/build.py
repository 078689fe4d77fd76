"""Compile oracle/sqeq_oracle.c into oracle/liboracle.so (gcc, fp64, OpenMP).

TEST INFRASTRUCTURE -- the oracle is never linked into or imported by the
product package.  `-ffp-contract=off` keeps every fp64 product and sum of the
cutoff predicate individually rounded (DESIGN.md R-NL); no -ffast-math.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sqeq_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        from . import cpu_method
        cpu_method.build()
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math",
           "-fopenmp", "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    from . import cpu_method            # the second CPU baseline (a restatement of the method, pinned against the oracle)
    cpu_method.build(force)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
