"""Builds oracle/libhomg_oracle.so from oracle/homg_oracle.cpp with g++.

ORACLE = TEST INFRASTRUCTURE.  Called by tests/conftest.py, __graft_entry__.build()
and bench.py's cpu_baseline / --impl reference legs; never by the product path.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "homg_oracle.cpp")
LIB = os.path.join(HERE, "libhomg_oracle.so")

# -ffp-contract=off: the compiler contracts nothing by itself, so the oracle's arithmetic is exactly the
# expression tree written in the source and a reader can check it by eye.  The only fused multiply-adds
# are the three explicit std::fma calls of the constant-coefficient Jacobi sweep (Eq. 3, R14).
CMD = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-ffp-contract=off", "-o", LIB, SRC]


def build(force: bool = False) -> str:
    """HOMG_ORACLE_CFLAGS (e.g. "-fsanitize=undefined -fno-sanitize-recover=all -g") adds flags for a one-off checked
    build (profiles/r02_sanitizer.md); such a build is always redone, and so is the next plain one."""
    extra = os.environ.get("HOMG_ORACLE_CFLAGS", "").split()
    stamp = LIB + ".flags"
    last = open(stamp).read() if os.path.exists(stamp) else ""
    if force or extra or last or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        subprocess.check_call(CMD[:-3] + extra + CMD[-3:])
        if extra:
            with open(stamp, "w") as fh:
                fh.write(" ".join(extra))
        elif os.path.exists(stamp):
            os.remove(stamp)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
