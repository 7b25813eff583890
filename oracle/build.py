"""Compile oracle/wl_oracle.c into oracle/libwl_oracle.so with gcc (-O2, OpenMP).

Test infrastructure: called by oracle/wl_oracle.py on first use and by
__graft_entry__.build().  No fast-math: the oracle's arithmetic is IEEE FP64.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "wl_oracle.c")
LIB = os.path.join(HERE, "libwl_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-D_GNU_SOURCE", "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
