"""Build the C-ABI library of include/nmpc.h with nvcc for sm_100a:

  libnmpc_b200.so        the product
  libnmpc_b200_aids.so   the same sources with -DNMPC_TRACE_BUILD (per-task timestamps in the persistent kernels) plus
                         csrc/peak.cu: measurement aids of include/nmpc_aids.h, never loaded by the product path

nvcc cross-compiles without a GPU, so this runs on the CPU-only container as well as on the B200 box.
Objects are rebuilt only when a source or header is newer than the object (in-tree `build/` directories).
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
BUILD_AIDS = os.path.join(HERE, "build", "aids")
LIB = os.path.join(HERE, "libnmpc_b200.so")
LIB_AIDS = os.path.join(HERE, "libnmpc_b200_aids.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC,-pthread", "-I", os.path.join(ROOT, "include")]
# (source, extra flags).  ipm.cu is built without FMA contraction so that its element-wise statements round like the
# plain fp64 expressions of the method; the dense kernels of factor.cu use FMA.
SOURCES = [
    ("symbolic.cpp", []),
    ("factor.cu", []),
    ("solve.cu", []),
    ("ipm.cu", ["-fmad=false"]),
    ("hykkt.cu", ["-fmad=false"]),
    ("api.cu", []),
]
AIDS_ONLY = [("peak.cu", [])]
HEADERS = ["device.h", "symbolic.h", "models.cuh", os.path.join(ROOT, "include", "nmpc.h"),
           os.path.join(ROOT, "include", "nmpc_aids.h")]


def _newest_header() -> float:
    t = 0.0
    for h in HEADERS:
        p = h if os.path.isabs(h) else os.path.join(CSRC, h)
        t = max(t, os.path.getmtime(p))
    return t


def _compile(src: str, extra: list[str], force: bool, hdr_t: float, bdir: str) -> tuple[str, bool]:
    s = os.path.join(CSRC, src)
    o = os.path.join(bdir, os.path.splitext(src)[0] + ".o")
    if not force and os.path.exists(o) and os.path.getmtime(o) >= max(os.path.getmtime(s), hdr_t):
        return o, False
    cmd = [NVCC] + ARCH + COMMON + extra + ["-c", s, "-o", o]
    subprocess.check_call(cmd)
    return o, True


def _link(lib: str, objs: list[str], verbose: bool) -> None:
    tmp = lib + f".tmp{os.getpid()}"
    subprocess.check_call([NVCC] + ARCH + ["-shared", "-o", tmp] + objs + ["-lcudart", "-lpthread"])
    os.replace(tmp, lib)
    if verbose:
        print("built", lib)


def build(force: bool = False, verbose: bool = False, aids: bool = True) -> str:
    os.makedirs(BUILD_AIDS, exist_ok=True)
    hdr_t = _newest_header()
    jobs = [(src, extra, BUILD) for src, extra in SOURCES]
    if aids:
        jobs += [(src, extra + ["-DNMPC_TRACE_BUILD"], BUILD_AIDS) for src, extra in SOURCES + AIDS_ONLY]
    with ThreadPoolExecutor(max_workers=6) as ex:
        res = list(ex.map(lambda a: _compile(a[0], a[1], force, hdr_t, a[2]), jobs))
    prod, aid = res[: len(SOURCES)], res[len(SOURCES):]
    if force or any(r[1] for r in prod) or not os.path.exists(LIB):
        _link(LIB, [r[0] for r in prod], verbose)
    if aids and (force or any(r[1] for r in aid) or not os.path.exists(LIB_AIDS)):
        _link(LIB_AIDS, [r[0] for r in aid], verbose)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
