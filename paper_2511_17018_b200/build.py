"""Builds libtpcclus.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2511_17018_b200.build [--force]

The kernel text (csrc/tpcclus_kernels.cuh) goes into the library twice: offline, cut into
compilation units that nvcc compiles one by one, in parallel, straight to GPU binaries
(PAPER.md 64; generic build, parameters in each unit's __constant__ block), and verbatim as a
string for the NVRTC build that create(TPCCLUS_RTC) performs (PAPER.md 91: "the source code is
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
GEN = os.path.join(GEN_DIR, "tpcclus_embedded.S")
SOURCES = [os.path.join(CSRC, "tpcclus.cu"), os.path.join(CSRC, "tpcclus_kernels.cuh"), os.path.join(CSRC, "tpcclus_unit.cu"),
           os.path.join(CSRC, "tpcclus_noalloc.cu"), os.path.join(ROOT, "include", "tpcclus.h")]

# compilation units (PAPER.md 64: one GPU binary per kernel family): name -> TPC_U_* bit of tpcclus_kernels.cuh
# (the units of reading Q10'' and the partition / debug units that feed them carry a time halo of 5: -DTPC_HALO=5u)
UNITS = {"part_coarse": (0x001, 3), "dir": (0x002, 3), "part_fine": (0x004, 3), "tiles_fast": (0x008, 3), "tiles_det": (0x010, 3),
         "order": (0x020, 3), "tiles_dump": (0x040, 3), "tiles_fast_g": (0x080, 3), "tiles_det_g": (0x100, 3),
         "part_coarse_h5": (0x001, 5), "part_fine_h5": (0x004, 5), "tiles_dump_h5": (0x040, 5),
         "tiles_fast_s": (0x200, 5), "tiles_det_s": (0x400, 5)}

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
DEVICE_FLAGS = [*ARCH, "-lineinfo", "-O3", "-std=c++17",
                "--fmad=false", "--prec-div=true", "--prec-sqrt=true", "--ftz=false"]   # PAPER.md 37-39
HOST_FLAGS = [*ARCH, "-O3", "-std=c++17", "-Xcompiler", "-fPIC,-fvisibility=hidden", "-shared", "-cudart", "static"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def unit_cubin(name: str) -> str:
    return os.path.join(GEN_DIR, "unit_%s.cubin" % name)


def _compile_unit(name: str, verbose: bool) -> str:
    """One unit straight to a GPU binary: nvcc -cubin for sm_100a (no PTX, no host code)."""
    out = unit_cubin(name)
    cmd = [_nvcc(), *DEVICE_FLAGS, *os.environ.get("TPC_EXTRA", "").split(), *(["-Xptxas", "-v"] if verbose else []),
           "-DTPC_UNITS=%du" % UNITS[name][0], "-DTPC_HALO=%du" % UNITS[name][1], "-cubin", "-o", out,
           os.path.join(CSRC, "tpcclus_unit.cu")]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed for unit %s:\n%s\n%s" % (name, r.stdout, r.stderr))
    return r.stderr


def _embed() -> None:
    """The unit binaries and the kernel text (for NVRTC; PAPER.md 91: "the source code is embedded in
    the library") go into the library through one assembler file of .incbin directives."""
    lines = ['.section .rodata', '.balign 16', '.global tpcclus_kernel_source', 'tpcclus_kernel_source:',
             '.incbin "%s"' % os.path.join(CSRC, "tpcclus_kernels.cuh"), '.byte 0']
    for name in UNITS:
        lines += ['.balign 16', '.global tpcclus_cubin_%s' % name, 'tpcclus_cubin_%s:' % name,
                  '.incbin "%s"' % unit_cubin(name), '.global tpcclus_cubin_%s_end' % name, 'tpcclus_cubin_%s_end:' % name]
    lines.append('.section .note.GNU-stack,"",@progbits')
    with open(GEN, "w") as f:
        f.write("\n".join(lines) + "\n")


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or older than a source. Returns the .so path."""
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(s) for s in SOURCES + [os.path.abspath(__file__)])
        if os.path.getmtime(LIB) >= newest:
            return LIB
    os.makedirs(GEN_DIR, exist_ok=True)
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as ex:   # PAPER.md 64: the units build in parallel
        logs = list(ex.map(lambda n: _compile_unit(n, verbose), UNITS))
    if verbose:
        for name, log in zip(UNITS, logs):
            print("== unit %s\n%s" % (name, log), file=sys.stderr)
    _embed()
    obj = os.path.join(GEN_DIR, "tpcclus_embedded.o")
    subprocess.check_call(["gcc", "-c", "-o", obj, GEN])
    # the handle-free entry point with its scratch in a static device array: an object of its own, device code for sm_100a
    noalloc = os.path.join(GEN_DIR, "tpcclus_noalloc.o")
    subprocess.check_call([_nvcc(), *DEVICE_FLAGS, "-Xcompiler", "-fPIC,-fvisibility=hidden", "-c", "-o", noalloc,
                           os.path.join(CSRC, "tpcclus_noalloc.cu")])
    tmp = LIB + ".tmp%d" % os.getpid()
    subprocess.check_call([_nvcc(), *HOST_FLAGS, *os.environ.get("TPC_EXTRA", "").split(), "-o", tmp, os.path.join(CSRC, "tpcclus.cu"), noalloc, obj, "-ldl"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
