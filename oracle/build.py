"""Build the CPU oracle (oracle/sp_oracle.c, oracle/ghg_oracle.c) into oracle/libsporacle.so with gcc.

Test infrastructure only: called by tests/, __graft_entry__.build() and bench.py's
cpu_baseline / --impl reference legs.  Building the checker is not using it.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sp_oracle.c")
SRC_GHG = os.path.join(HERE, "ghg_oracle.c")
LIB = os.path.join(HERE, "libsporacle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(SRC_GHG)):
        return LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", LIB, SRC, SRC_GHG, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
