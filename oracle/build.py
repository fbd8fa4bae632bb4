"""Build the oracle shared library (test infrastructure; see ipa_oracle.cpp header).

    python oracle/build.py          # -> oracle/libipa_oracle.so

Plain g++ -O2, no -ffast-math (the oracle is timed as it stands).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ipa_oracle.cpp")
LIB = os.path.join(HERE, "libipa_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
