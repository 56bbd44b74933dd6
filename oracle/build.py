"""Build the oracle shared library (test infrastructure; gcc only).

Flags recorded in DESIGN.md: -O2 -ffp-contract=off so that no multiply-add is
contracted except the fma() calls the source writes; -mfma only makes those
explicit calls hardware instructions (same correctly-rounded result).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mcdc_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")


def build(force=False):
    # ORACLE_LIB: a library built by hand from the same source (e.g. with -fsanitize=address,undefined) to run the
    # CPU test suite under a sanitizer: LD_PRELOAD=$(gcc -print-file-name=libasan.so) ORACLE_LIB=... pytest -m "not gpu"
    if os.environ.get("ORACLE_LIB"):
        return os.environ["ORACLE_LIB"]
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC),
                                             os.path.getmtime(os.path.join(HERE, "mcdc_oracle.h")))):
        return LIB
    cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-math-errno", "-mfma",
           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
