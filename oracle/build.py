"""Build the CPU oracle (TEST INFRASTRUCTURE ONLY) into oracle/libqcd_oracle.so.

Plain g++ -O2 -fopenmp, no -ffast-math.  Building the checker is not using it:
__graft_entry__.build() calls this; the product never loads the result.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "qcd_oracle.cpp")
LIB = os.path.join(HERE, "libqcd_oracle.so")
ON_SRC = os.path.join(HERE, "on_oracle.cpp")       # the O(N) model oracle
ON_LIB = os.path.join(HERE, "libqcd_on_oracle.so")


def build_oracle(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


def build_on_oracle(force: bool = False) -> str:
    if not force and os.path.exists(ON_LIB) and os.path.getmtime(ON_LIB) >= os.path.getmtime(ON_SRC):
        return ON_LIB
    subprocess.run(["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", ON_LIB, ON_SRC], check=True)
    return ON_LIB


if __name__ == "__main__":
    print(build_oracle(force=True))
    print(build_on_oracle(force=True))
