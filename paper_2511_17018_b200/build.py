"""Builds libtpcclus.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2511_17018_b200.build [--force]

The kernel text (csrc/tpcclus_kernels.cuh) is compiled twice into the library: offline by
nvcc (generic build, parameters in __constant__ memory) and embedded verbatim as a string
for the NVRTC build that create(TPCCLUS_RTC) performs (PAPER.md 91: "the source code is
embedded in the library").
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtpcclus.so")
GEN_DIR = os.path.join(ROOT, "build")
GEN = os.path.join(GEN_DIR, "tpcclus_kernel_source.c")
SOURCES = [os.path.join(CSRC, "tpcclus.cu"), os.path.join(CSRC, "tpcclus_kernels.cuh"),
           os.path.join(ROOT, "include", "tpcclus.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "--fmad=false", "--prec-div=true", "--prec-sqrt=true", "--ftz=false",   # PAPER.md 37-39
    "-Xcompiler", "-fPIC,-fvisibility=hidden", "-shared", "-cudart", "static",
]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _embed_source() -> None:
    os.makedirs(GEN_DIR, exist_ok=True)
    with open(os.path.join(CSRC, "tpcclus_kernels.cuh"), "rb") as f:
        src = f.read()
    text = "const char tpcclus_kernel_source[] = {" + ",".join(str(b) for b in src) + ",0};\n"
    with open(GEN, "w") as f:
        f.write(text)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or older than a source. Returns the .so path."""
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(s) for s in SOURCES + [os.path.abspath(__file__)])
        if os.path.getmtime(LIB) >= newest:
            return LIB
    _embed_source()
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = [_nvcc(), *NVCC_FLAGS, *os.environ.get("TPC_EXTRA", "").split(), *(["-Xptxas", "-v"] if verbose else []), "-o", tmp,
           os.path.join(CSRC, "tpcclus.cu"), GEN, "-ldl"]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
