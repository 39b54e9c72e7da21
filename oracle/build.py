"""Build the CPU oracle shared library (TEST INFRASTRUCTURE ONLY).

    python -m oracle.build        -> oracle/libmkv_oracle.so

gcc flags: -O2, no -ffast-math, -ffp-contract=off (O1/O2 fix an fp32 operation order),
-fopenmp (parallel over independent units only).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mkv_oracle.c")
HDR = os.path.join(HERE, "mkv_oracle.h")
LIB = os.path.join(HERE, "libmkv_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        if os.path.getmtime(LIB) >= newest:
            return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-ffp-contract=off", "-fno-fast-math",
           "-fopenmp", "-shared", "-fPIC", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
