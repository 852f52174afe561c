"""Build libgcorbit.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo snapshot).  The
bench-side microbenchmarks (libgcprobes.so) are built by bench_probes/probes.py, outside this package."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
SO = os.path.join(_HERE, "libgcorbit.so")
SOURCES = ["gcorbit_api.cu"]
HEADERS = ["device_math.cuh", "field.cuh", "kernels_generic.cuh", "kernels_grid.cuh", "kernels_lane.cuh", "kernels_symplectic.cuh", "kernels_warp.cuh", "kernels_tile.cuh", "kernels_mma.cuh",
           os.path.join("..", "..", "include", "gcorbit.h")]


def nvcc_cmd(extra=(), sources=None, out=None):
    return ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
            "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v", *extra,
            *[os.path.join(CSRC, s) for s in (sources or SOURCES)], "-o", out or SO]


STAMP = SO + ".srchash"


def source_hash() -> str:
    """Content hash of everything the library is built from (mtimes do not survive a repo snapshot)."""
    import hashlib
    h = hashlib.sha256()
    for d in [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]:
        with open(d, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def needs_build() -> bool:
    if not os.path.exists(SO) or not os.path.exists(STAMP):
        return True
    with open(STAMP) as fh:
        return fh.read().strip() != source_hash()


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    if force or needs_build():
        r = subprocess.run(nvcc_cmd(extra), capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed building libgcorbit.so")
        with open(os.path.join(_HERE, "build_ptxas.log"), "w") as fh:
            fh.write(" ".join(nvcc_cmd(extra)) + "\n" + r.stdout + r.stderr)
        with open(STAMP, "w") as fh:
            fh.write(source_hash())
    return SO


if __name__ == "__main__":
    build(force=True, verbose=True, extra=tuple(sys.argv[1:]))
