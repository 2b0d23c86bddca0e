"""Build oracle/liboracle.so with gcc (plain C, no FMA contraction).  TEST INFRASTRUCTURE.

    python -m oracle.build          # or: python oracle/build.py
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "md_oracle.c")
SRC_EXT = os.path.join(HERE, "md_oracle_ext.c")  # virial, further force fields
LIB = os.path.join(HERE, "liboracle.so")
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-std=c11", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(SRC), os.path.getmtime(SRC_EXT))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest:
        return LIB
    cmd = ["gcc", *CFLAGS, "-o", LIB, SRC, SRC_EXT, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
