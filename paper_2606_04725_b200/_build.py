"""Build paper_2606_04725_b200/libnmpc_b200.so (the C-ABI library of include/nmpc.h) with nvcc for sm_100a.

nvcc cross-compiles without a GPU, so this runs on the CPU-only container as well as on the B200 box.
Objects are rebuilt only when a source or header is newer than the object (in-tree `build/` directory).
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
BUILD = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libnmpc_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include")]
# (source, extra flags).  ipm.cu is built without FMA contraction so that its element-wise statements round like the
# plain fp64 expressions of the method; the dense kernels of factor.cu use FMA.
SOURCES = [
    ("symbolic.cpp", []),
    ("factor.cu", []),
    ("solve.cu", []),
    ("ipm.cu", ["-fmad=false"]),
    ("api.cu", []),
    ("peak.cu", []),
]
HEADERS = ["device.h", "symbolic.h", "models.cuh", os.path.join(ROOT, "include", "nmpc.h")]


def _newest_header() -> float:
    t = 0.0
    for h in HEADERS:
        p = h if os.path.isabs(h) else os.path.join(CSRC, h)
        t = max(t, os.path.getmtime(p))
    return t


def _compile(src: str, extra: list[str], force: bool, hdr_t: float) -> tuple[str, bool]:
    s = os.path.join(CSRC, src)
    o = os.path.join(BUILD, os.path.splitext(src)[0] + ".o")
    if not force and os.path.exists(o) and os.path.getmtime(o) >= max(os.path.getmtime(s), hdr_t):
        return o, False
    cmd = [NVCC] + ARCH + COMMON + extra + ["-c", s, "-o", o]
    subprocess.check_call(cmd)
    return o, True


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(BUILD, exist_ok=True)
    hdr_t = _newest_header()
    with ThreadPoolExecutor(max_workers=4) as ex:
        res = list(ex.map(lambda a: _compile(a[0], a[1], force, hdr_t), SOURCES))
    objs = [r[0] for r in res]
    if force or any(r[1] for r in res) or not os.path.exists(LIB):
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call([NVCC] + ARCH + ["-shared", "-o", tmp] + objs + ["-lcudart"])
        os.replace(tmp, LIB)
        if verbose:
            print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
