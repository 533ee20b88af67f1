"""Build the CPU oracle (oracle/libmdwf_oracle.so) with gcc.  TEST INFRASTRUCTURE ONLY.

Building the checker is not using it: __graft_entry__.build() calls this, the product
path (paper_1701_07559_b200/) never loads the result.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mdwf_oracle.c")
LIB = os.path.join(HERE, "libmdwf_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
