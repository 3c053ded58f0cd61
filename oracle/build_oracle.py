"""Build the CPU oracle (test infrastructure) into oracle/libsfd_oracle.so with g++.

Called by __graft_entry__.build(), tests/conftest.py and bench.py's cpu_baseline leg.
Building the checker is not using it: nothing under paper_2304_06340_b200/ links or loads it.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "sfd_oracle.cpp"), os.path.join(HERE, "sfd_oracle_exact.cpp")]
LIB = os.path.join(HERE, "libsfd_oracle.so")
# -lquadmath: sfd_oracle_exact.cpp evaluates the exact triangle transform (eq. 2.19) in binary128
CMD = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", *SRCS, "-o", LIB, "-lquadmath"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(s) for s in SRCS):
        subprocess.run(CMD, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
