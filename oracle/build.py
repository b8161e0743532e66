"""oracle/build.py — compiles the CPU ORACLE (test infrastructure, not the product).

`build()` runs gcc on oracle/nfs_oracle.c and leaves oracle/libnfs_oracle.so beside it.
No -ffast-math: the oracle is the plain fp64 definition.
"""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "nfs_oracle.c")
LIB = os.path.join(_HERE, "libnfs_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["gcc", "-O2", "-fopenmp", "-fno-fast-math", "-shared", "-fPIC", "-o", tmp, SRC, "-lm"]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
