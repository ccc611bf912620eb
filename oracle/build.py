"""oracle/build.py -- TEST INFRASTRUCTURE.  Compiles the CPU oracle into oracle/liblbr_oracle.so.

g++ -O2 -ffp-contract=off (no fused multiply-adds: the status decision must use plain IEEE
operations) with OpenMP and libquadmath.  Called by __graft_entry__.build() and,
lazily, by oracle/pyoracle.py.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SO = os.path.join(HERE, "liblbr_oracle.so")
SOURCES = [os.path.join(HERE, "oracle_capi.cpp"), os.path.join(HERE, "opcount.cpp")]
DEPS = SOURCES + [os.path.join(HERE, "lbr_oracle.hpp")]


def build(force: bool = False) -> str:
    if not force and os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(d) for d in DEPS):
        return SO
    cmd = ["g++", "-std=gnu++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-fopenmp",
           "-o", SO] + SOURCES + ["-lquadmath", "-lm"]
    subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force=True))
