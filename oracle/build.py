"""Build the CPU oracle shared library (TEST INFRASTRUCTURE ONLY; see mlcc_oracle.c)."""
import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
STAMP = LIB + ".host"
SOURCES = [os.path.join(HERE, "mlcc_oracle.c"), os.path.join(HERE, "aberth_generic.inc")]
FLAGS = ["-O3", "-march=native", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra"]


def _host_signature() -> str:
    """-march=native ties the library to the CPU it was built on: the in-tree .so also travels to other boxes, so the
    build host's instruction-set flags are kept beside it and a different host rebuilds."""
    flags = ""
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("flags"):
                flags = line
                break
    except OSError:
        pass
    return hashlib.sha1((flags + " ".join(FLAGS)).encode()).hexdigest()


def build(force: bool = False) -> str:
    """gcc -O3 -march=native -ffp-contract=off -fopenmp -> oracle/liboracle.so; returns its path.  The arithmetic is the
    same as with -O2: contraction is off and gcc does not reassociate floating-point sums without -ffast-math."""
    sig = _host_signature()
    if not force and os.path.exists(LIB) and os.path.exists(STAMP) and open(STAMP).read().strip() == sig:
        if all(os.path.getmtime(LIB) >= os.path.getmtime(s) for s in SOURCES):
            return LIB
    cmd = ["gcc", *FLAGS, "-o", LIB, SOURCES[0], "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    with open(STAMP, "w") as f:
        f.write(sig + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force=True))
