"""ctypes binding of libgcprobes.so (bench_probes/fp64_probes.cu): microbenchmarks of the box that bench.py reports beside
its roofline (DFMA rate, DMMA.8x8x4 rate alone and mixed with DFMA, LDS.128 issue cost).  Bench-side only: none of
this is part of the product boundary (include/gcorbit.h) or of libgcorbit.so."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "libgcprobes.so")
EXPORTS = ["gcprobe_dfma", "gcprobe_dmma", "gcprobe_lds128"]
SRC = os.path.join(_HERE, "fp64_probes.cu")
_lib = None


def build(force: bool = False) -> str:
    """nvcc for sm_100a, in-tree (the .so travels with the repo snapshot); rebuilt when the source is newer or the
    recorded content hash differs (mtimes do not survive a snapshot)."""
    import hashlib
    with open(SRC, "rb") as fh:
        digest = hashlib.sha256(fh.read()).hexdigest()
    stamp = SO_PATH + ".srchash"
    if not force and os.path.exists(SO_PATH) and os.path.exists(stamp) and open(stamp).read().strip() == digest:
        return SO_PATH
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared",
           "-Xcompiler", "-fPIC", SRC, "-o", SO_PATH]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed building libgcprobes.so")
    with open(stamp, "w") as fh:
        fh.write(digest)
    return SO_PATH


def load_library():
    global _lib
    if _lib is None:
        if not os.path.exists(SO_PATH):
            raise FileNotFoundError(f"{SO_PATH} not built: run `python __graft_entry__.py build`")
        L = C.CDLL(SO_PATH)
        for name in EXPORTS:
            fn = getattr(L, name)
            fn.restype = C.c_int
            fn.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double)]
        _lib = L
    return _lib


def _pair(name):
    a, b = C.c_double(0), C.c_double(0)
    rc = getattr(load_library(), name)(C.byref(a), C.byref(b))
    if rc != 0:
        raise RuntimeError(f"{name}: CUDA error {rc}")
    return a.value, b.value


def dfma():
    """(FP64 FLOP/s of a register-only DFMA loop, elapsed ms)."""
    return _pair("gcprobe_dfma")


def dmma():
    """(DMMA.8x8x4 alone, DMMA + DFMA mixed) in FLOP/s."""
    return _pair("gcprobe_dmma")


def lds128():
    """SM cycles per warp-wide LDS.128: (all lanes distinct 16-byte addresses, lane pairs sharing 16 bytes)."""
    return _pair("gcprobe_lds128")
