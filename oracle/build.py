"""Compile oracle/oscnet_oracle.c into oracle/liboscnet_oracle.so with gcc.

Building the checker is not using it: ``__graft_entry__.build()`` calls
``build()`` here so that the GPU box has the shared object.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "oscnet_oracle.c")
LIB = os.path.join(HERE, "liboscnet_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    # -O2, no -ffast-math: the oracle's arithmetic is exactly what is written.
    # (written beside and renamed into place: a process that has the old object mapped keeps it)
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp",
           "-ffp-contract=off", SRC, "-o", tmp, "-lm"]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
