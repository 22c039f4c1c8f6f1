"""Build oracle/libaptsig_oracle.so with gcc (test infrastructure; see aptsig_oracle.c header)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "aptsig_oracle.c")
LIB = os.path.join(HERE, "libaptsig_oracle.so")
FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-Wall"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        subprocess.check_call(["gcc", *FLAGS, SRC, "-o", LIB, "-lm"])
    return LIB


if __name__ == "__main__":
    print(build(force=True))
