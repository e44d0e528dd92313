"""Build the CPU oracle (test infrastructure) into oracle/liboracle.so with g++ -O2 -fopenmp (no fast-math)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cales_oracle.cpp")
LIB = os.path.join(HERE, "liboracle.so")


def build(force: bool = False) -> str:
    if os.environ.get("CALES_ORACLE_LIB"):      # tests/test_oracle_mutants.py points the binding at a deliberately broken build
        return os.environ["CALES_ORACLE_LIB"]
    deps = [SRC, os.path.join(HERE, "cales_oracle.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wno-misleading-indentation",
           "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
