"""Build the fp64 CPU oracle (test infrastructure) into oracle/libpd_oracle.so with gcc.

Usage: python -m oracle.build   (also called by __graft_entry__.build(), tests/conftest.py and
bench.py's cpu_baseline leg).  Building the checker is not using it: the product path never loads
this library.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pd_oracle.c")
HDR = os.path.join(HERE, "pd_oracle.h")
LIB = os.path.join(HERE, "libpd_oracle.so")

# -ffp-contract=off: no fused multiply-add, so the arithmetic is the formula as written.
CFLAGS = ["-O2", "-ffp-contract=off", "-std=c99", "-Wall", "-Wextra", "-shared", "-fPIC"]


def build(force: bool = False) -> str:
    """Compile if the library is missing or older than its sources; return its path."""
    stale = (
        force
        or not os.path.exists(LIB)
        or os.path.getmtime(LIB) < max(os.path.getmtime(SRC), os.path.getmtime(HDR))
    )
    if stale:
        tmp = LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, SRC, "-lm"])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
