"""Builds the C-ABI CUDA library (libpsc_b200.so) in-tree with nvcc for sm_100a.

    python -m paper_1310_7866_b200.build [--force]

nvcc cross-compiles without a GPU.  The library links the CUDA runtime statically, so it does
not depend on which libcudart PyTorch ships.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(_ROOT, "include")
LIB = os.path.join(_HERE, "libpsc_b200.so")
SOURCES = ["api.cu", "fields.cu", "sort.cu", "push1.cu", "push2.cu", "marder.cu", "balance.cu"]
HEADERS = ["psc_internal.cuh", "push_common.cuh", "store.cuh"]

COMMON = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17", "--extended-lambda", "-Xcompiler", "-fPIC",
]
# sort.cu launches kernels from the device (the re-layout gate): relocatable device code + device link
RDC_SOURCES = ["sort.cu"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: the CUDA library cannot be built (there is no CPU fallback)")


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(INCLUDE, "psc.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if the library is missing or older than its sources.  Returns its path."""
    if not force and not _stale():
        return LIB
    from concurrent.futures import ThreadPoolExecutor

    nvcc = _nvcc()
    bdir = os.path.join(_HERE, "build", "obj.%d" % os.getpid())
    os.makedirs(bdir, exist_ok=True)
    inc = ["-I", INCLUDE, "-I", CSRC]
    vflags = ["-Xptxas", "-v"] if verbose else []

    def compile_one(f):
        obj = os.path.join(bdir, f.replace(".cu", ".o"))
        mode = ["-dc"] if f in RDC_SOURCES else ["-c"]
        subprocess.check_call([nvcc] + COMMON + vflags + mode + inc + ["-o", obj, os.path.join(CSRC, f)])
        return obj

    try:
        with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
            objs = list(ex.map(compile_one, SOURCES))
        rdc_objs = [o for o, f in zip(objs, SOURCES) if f in RDC_SOURCES]
        dlink = os.path.join(bdir, "dlink.o")
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-Xcompiler", "-fPIC",
                               "-dlink", "-o", dlink] + rdc_objs + ["-lcudadevrt"])
        tmp = LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static",
                               "-o", tmp] + objs + [dlink, "-lcudadevrt"])
        os.replace(tmp, LIB)
    finally:
        shutil.rmtree(bdir, ignore_errors=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
