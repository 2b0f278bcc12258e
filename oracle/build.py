"""Build the CPU oracle shared library (test infrastructure).  `python -m oracle.build`."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sd_mhd_oracle.cpp")
LIB = os.path.join(HERE, "libsd_mhd_oracle.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "sd_mhd_oracle.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    # -ffp-contract=off: no FMA contraction, so the arithmetic is exactly what the source says.
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
           "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
