"""Compile oracle/debye_oracle.c into oracle/liboracle_debye.so with gcc (test infrastructure only)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "debye_oracle.c")
OUT = os.path.join(HERE, "liboracle_debye.so")


def build(force: bool = False) -> str:
    if force or not os.path.exists(OUT) or os.path.getmtime(OUT) < os.path.getmtime(SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=gnu11", "-o", OUT, SRC, "-lm"])
    return OUT


if __name__ == "__main__":
    print(build(force=True))
