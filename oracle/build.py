"""Build the CPU oracle shared library (test infrastructure only; see sht_oracle.cpp header).

    python oracle/build.py            # -> oracle/libsht_oracle.so
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sht_oracle.cpp")
OUT = os.path.join(HERE, "libsht_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(OUT) and os.path.getmtime(OUT) >= os.path.getmtime(SRC):
        return OUT
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", OUT, SRC, "-lm"]
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
