"""Compile the C oracle into oracle/librpa_oracle.so (plain gcc, OpenMP, no -march so the .so is portable
between the build box and the GPU box).  Building the checker is not using it: only tests/, smoke() and
bench.py's cpu_baseline / --impl reference legs load the result."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "rpa_oracle.c")
LIB = os.path.join(HERE, "librpa_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
