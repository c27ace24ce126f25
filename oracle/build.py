"""Build the CPU oracle (test infrastructure) into oracle/liboracle.so with g++ -O2 -fopenmp (no fast-math)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "wpcd_oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-o", LIB, SRC]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
