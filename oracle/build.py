"""Build the CPU oracle shared library (test infrastructure; see su_oracle.h).

    python oracle/build.py            # -> oracle/liboracle.so

-ffp-contract=off: the oracle evaluates the formulas as written (no FMA contraction), R19.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "su_oracle.cpp")
# SU_ORACLE_SANITIZE=1: the same source with AddressSanitizer + UndefinedBehaviorSanitizer (liboracle_san.so), for
#   SU_ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 python -m pytest tests -m "not gpu"
SANITIZE = os.environ.get("SU_ORACLE_SANITIZE", "") not in ("", "0")
LIB = os.path.join(HERE, "liboracle_san.so" if SANITIZE else "liboracle.so")
FLAGS = ["-O2", "-fopenmp", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-Wall"]
if SANITIZE:
    FLAGS += ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "su_oracle.h")]
    if (not force and os.path.exists(LIB)
            and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps)):
        return LIB
    cmd = ["g++", *FLAGS, "-o", LIB, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
