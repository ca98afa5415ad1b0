"""Build the oracle's C file into oracle/libfdas_oracle.so (gcc, OpenMP).  TEST INFRASTRUCTURE.

Run as `python oracle/build.py` or call `build()`.  The library is rebuilt when the source is newer
than the shared object.  Building the checker is not using it: `__graft_entry__.build()` calls this.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "fdas_oracle.c")
LIB = os.path.join(HERE, "libfdas_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # -O2 -ftree-vectorize without -ffast-math: the sums keep the order written in the source.
    cmd = ["gcc", "-O2", "-ftree-vectorize", "-fopenmp", "-fPIC", "-shared", "-std=c11",
           "-Wall", "-Wextra", "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
