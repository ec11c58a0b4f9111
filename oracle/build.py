"""Build the ORACLE shared library (test infrastructure, not the product).

    python -m oracle.build        # -> oracle/libsc_oracle.so

gcc -O2 -ffp-contract=off: no FMA contraction, so the deposit's index/fraction arithmetic is the
literal IEEE sequence written in sc_oracle.c.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sc_oracle.c")
LIB = os.path.join(HERE, "libsc_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(os.path.join(HERE, "sc_oracle.h")))):
        return LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-std=c99", "-Wall", "-Wextra", "-fPIC", "-shared",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
