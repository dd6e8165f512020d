"""Compile the CPU oracle (oracle/pd_oracle.cpp) into oracle/libpd_oracle.so with g++ -O2.

Test infrastructure only: building the checker is not using it (the product never loads it).
Usage: python oracle/build.py [--force]
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pd_oracle.cpp")
HDR = os.path.join(HERE, "pd_oracle.h")
LIB = os.path.join(HERE, "libpd_oracle.so")


def build(force: bool = False) -> str:
    """Build (if stale) and return the path of libpd_oracle.so."""
    if not force and os.path.exists(LIB):
        newest_src = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        if os.path.getmtime(LIB) >= newest_src:
            return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["g++", "-std=c++17", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(tmp, LIB)  # atomic: concurrent test workers never see a half-written library
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
