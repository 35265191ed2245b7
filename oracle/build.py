"""Compile the CPU oracle (oracle/bzo.c -> oracle/libbzo.so) with gcc.

TEST INFRASTRUCTURE: the product (paper_1912_04457_b200) never imports this package.
-ffp-contract=off: every + - * / sqrt of the sample generation rounds separately.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "bzo.c")
LIB = os.path.join(HERE, "libbzo.so")
FLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"]


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "bzo.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.run(["gcc", *FLAGS, SRC, "-o", tmp, "-lm"], check=True, cwd=HERE)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
