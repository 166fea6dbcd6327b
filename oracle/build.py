"""Build the CPU oracle (test infrastructure) into oracle/liblattice_oracle.so.

g++ -O2 -std=c++17 -ffp-contract=off -fopenmp -shared -fPIC.  Called by __graft_entry__.build()
and lazily by oracle/__init__.py; building the checker is not using it."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lattice_oracle.cpp")
LIB = os.path.join(HERE, "liblattice_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
           "-Wall", "-Wextra", "-o", LIB + ".tmp", SRC]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
