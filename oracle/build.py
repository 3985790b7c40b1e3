"""Build the CPU oracle (plain C, fp64) into oracle/libabm_oracle.so.

TEST INFRASTRUCTURE.  Compiled with strict IEEE semantics: no -ffast-math, no FMA contraction,
no -march flags, so the arithmetic is exactly what oracle/abm_oracle.c spells out.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "abm_oracle.c")
HDR = os.path.join(HERE, "abm_oracle.h")
LIB = os.path.join(HERE, "libabm_oracle.so")


def build(force: bool = False) -> str:
    newest_src = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= newest_src:
        return LIB
    cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
