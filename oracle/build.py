"""Build the CPU oracle (test infrastructure) into oracle/libstreams_oracle.so.

gcc -O2 -ffp-contract=off keeps every product and sum individually rounded, so the
oracle's arithmetic is exactly what streams_oracle.c spells out (A19).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "streams_oracle.c")
LIB = os.path.join(HERE, "libstreams_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(SRC[:-2] + ".h"))):
        return LIB
    cmd = ["gcc", "-std=gnu11", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-Wall",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
