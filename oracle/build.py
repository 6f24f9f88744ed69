"""Build the CPU oracle (test infrastructure) into oracle/libcap_oracle.so.

gcc -O2 -std=c11 -ffp-contract=off: no FMA contraction, so every fp32 step in
cap_oracle.c is a single IEEE operation (the explicit fmaf() calls excepted).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cap_oracle.c")
LIB = os.path.join(HERE, "libcap_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
