"""Compile the CPU oracle (oracle/heom_oracle.cpp) into oracle/libheom_oracle.so.

Building the checker is not using it: `__graft_entry__.build()` calls this, the
product never loads the result.  Plain g++, OpenMP for the loop over nodes.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "heom_oracle.cpp")
HDR = os.path.join(HERE, "heom_oracle.h")
LIB = os.path.join(HERE, "libheom_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fcx-limited-range", "-Wall", "-Wextra",
           "-shared", "-fPIC", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
