"""Build the CPU oracle (test infrastructure) with g++.

    python oracle/build.py

Writes oracle/libmonc_adv_oracle.so next to this file.  -ffp-contract=off keeps
the evaluation order written in monc_adv_oracle.cpp (no FMA contraction), so the
oracle is reproducible across compilers (SURVEY.md 8(c).2 "Oracle evaluation
order").  OpenMP is used only to split the outer x loop; results do not depend
on the thread count.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "monc_adv_oracle.cpp")
LIB = os.path.join(HERE, "libmonc_adv_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
