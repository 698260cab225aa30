"""Build the CPU oracle (test infrastructure) into oracle/librosen_oracle.so with g++.

Flags: -O2 -ffp-contract=off so that gcc never fuses a multiply and an add on its own; every
fused operation of the real-space path is an explicit std::fmaf.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SOURCES = ["rosen_oracle.cpp", "saw_enum.cpp"]
TARGET = os.path.join(HERE, "librosen_oracle.so")


def build(force: bool = False) -> str:
    srcs = [os.path.join(HERE, s) for s in SOURCES]
    if not force and os.path.exists(TARGET):
        if all(os.path.getmtime(TARGET) >= os.path.getmtime(s) for s in srcs):
            return TARGET
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-Wall", "-Wextra",
           "-shared", "-fPIC", "-o", TARGET] + srcs
    subprocess.run(cmd, check=True)
    return TARGET


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
