"""Build the CPU oracle (TEST INFRASTRUCTURE ONLY -- see dslash_oracle.c header).

    python oracle/build.py        # -> oracle/libdslash_oracle.so

Plain gcc; no CUDA, no torch, nothing from paper_2301_03636_b200/.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "dslash_oracle.c")
LIB = os.path.join(HERE, "libdslash_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c99", "-fcx-limited-range", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
