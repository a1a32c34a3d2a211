"""Compile oracle/chol.c into oracle/liborc_chol.so with gcc (test infrastructure; see oracle/__init__.py)."""
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(_HERE, "liborc_chol.so")
SRC = os.path.join(_HERE, "chol.c")


def build(force: bool = False) -> str:
    if force or (not os.path.exists(LIB)) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-std=c99", "-o", tmp, SRC, "-lm"])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
