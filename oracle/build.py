"""Build the CPU oracle shared library (TEST INFRASTRUCTURE ONLY; see mlcc_oracle.c)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
SOURCES = [os.path.join(HERE, "mlcc_oracle.c"), os.path.join(HERE, "aberth_generic.inc")]


def build(force: bool = False) -> str:
    """gcc -O2 -ffp-contract=off -fopenmp -> oracle/liboracle.so; returns its path."""
    if not force and os.path.exists(LIB):
        if all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in SOURCES):
            return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SOURCES[0], "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
