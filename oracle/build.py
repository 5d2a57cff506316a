"""Build the C oracle (oracle/cheb_oracle.c -> oracle/libcheb_oracle.so) with gcc.

Building the checker is not using it: __graft_entry__.build() calls this; the product never
loads the result.  Plain -O2, no -ffast-math (the oracle's arithmetic must stay IEEE).
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcheb_oracle.so")
SRC_PATH = os.path.join(_HERE, "cheb_oracle.c")


def build(verbose: bool = False) -> str:
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall",
           "-o", LIB_PATH, SRC_PATH, "-lm"]
    if verbose:
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    return LIB_PATH


if __name__ == "__main__":
    build(verbose=True)
