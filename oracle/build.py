"""Build the CPU oracle shared library (test infrastructure, not the product).

g++ -O2 -ffp-contract=off -fopenmp: no fast-math, no FMA contraction, so every formula of
fvnl_oracle.cpp rounds exactly as written.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "fvnl_oracle.cpp")
# FVNL_ORACLE_VARIANT=fma: the SAME source compiled with FMA contraction allowed -- a second CPU program that differs from the
# oracle by rounding only.  Used by tests/golden/make_c4_sensitivity.py alone, to measure how far two roundings of the scheme
# drift apart on a workload; never the reference of a parity test.
VARIANT = os.environ.get("FVNL_ORACLE_VARIANT", "")
assert VARIANT in ("", "fma"), VARIANT
LIB = os.path.join(HERE, "libfvnl_oracle_fma.so" if VARIANT else "libfvnl_oracle.so")
CONTRACT = ["-ffp-contract=fast", "-mfma"] if VARIANT else ["-ffp-contract=off"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = f"{LIB}.{os.getpid()}.tmp"                  # appear atomically: a running process keeps its mapped copy
    cmd = ["g++", "-std=c++17", "-O2"] + CONTRACT + ["-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-o", tmp, SRC]
    try:
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    finally:
        if os.path.exists(tmp):
            os.remove(tmp)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
