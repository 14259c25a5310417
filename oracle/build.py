"""Build the fp64 CPU oracle (oracle/haste_oracle.cpp) into oracle/libhaste_oracle.so.

TEST INFRASTRUCTURE, not the product.  `python oracle/build.py` or `build()`;
`__graft_entry__.build()` calls it too (building the checker is not using it).
"""
import os
import subprocess

_DIR = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_DIR, "haste_oracle.cpp")
LIB = os.path.join(_DIR, "libhaste_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
