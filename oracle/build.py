"""Build the CPU oracle shared library (test infrastructure only; see lgf_oracle.cpp header).

    python oracle/build.py        ->  oracle/liblgf_oracle.so
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lgf_oracle.cpp")
OUT = os.path.join(HERE, "liblgf_oracle.so")
FLAGS = ["-O2", "-fopenmp", "-shared", "-fPIC", "-std=c++17", "-ffp-contract=off"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(OUT) and os.path.getmtime(OUT) >= os.path.getmtime(SRC):
        return OUT
    cmd = ["g++"] + FLAGS + [SRC, "-o", OUT]
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
