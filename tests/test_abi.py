"""CPU-side checks of the boundary: libgcorbit.so builds for sm_100a, loads without a GPU, exports every
symbol include/gcorbit.h declares, validates its arguments before touching a device, and fails loudly -- never
falls back -- when no CUDA device is present."""
from __future__ import annotations

import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2605_16734_b200 import build, gcorbit
    build.build()
    return gcorbit.load_library()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "gcorbit.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gc_[a-z0-9_]+)\s*\(", text)))


def test_header_and_library_agree(lib):
    from paper_2605_16734_b200 import gcorbit
    names = declared_functions()
    assert "gc_trace" in names and "gc_field_create" in names and len(names) >= 11
    assert sorted(gcorbit.EXPORTS) == names
    for nm in names:
        assert getattr(lib, nm) is not None


def test_boundary_holds_the_method_only():
    """The product library exports the calls of the method and nothing else: the FP64 / shared-memory
    microbenchmarks bench.py reports live in bench_probes/libgcprobes.so (bench-side, outside the package), not behind
    include/gcorbit.h."""
    import subprocess
    from paper_2605_16734_b200 import build
    from bench_probes import probes
    probes.build()
    syms = subprocess.run(["nm", "-D", "--defined-only", build.SO], capture_output=True, text=True).stdout
    exported = sorted(set(re.findall(r"\bT (gc[a-z0-9_]*)", syms)))
    assert exported == declared_functions(), exported
    plib = probes.load_library()
    for nm in probes.EXPORTS:
        assert getattr(plib, nm) is not None


def test_library_is_sm100a_native():
    """The cubin inside the library targets sm_100a and nothing else (no PTX JIT, no other arch)."""
    import subprocess
    from paper_2605_16734_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.SO], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_struct_layouts_match_the_header():
    from paper_2605_16734_b200 import gcorbit
    # gc_trace_params: 11 doubles + 3 int64; gc_field_desc: pointers and int32 with natural alignment
    assert C.sizeof(gcorbit.gc_trace_params) == 11 * 8 + 3 * 8
    assert C.sizeof(gcorbit.gc_field_desc) == 16 + 6 * 8 + 8 + 8 + 5 * 8 + 3 * 8          # + bmns, kmnc, kmns (NEXT-4)
    assert gcorbit.gc_field_desc.psi0.offset == 64 and gcorbit.gc_field_desc.nk.offset == 72


def _desc(fld, **over):
    from paper_2605_16734_b200 import gcorbit as G
    k = dict(xm=np.ascontiguousarray(fld.xm, np.int32), xn=np.ascontiguousarray(fld.xn, np.int32),
             bmnc=np.ascontiguousarray(fld.bmnc), G=np.ascontiguousarray(fld.G), I=np.ascontiguousarray(fld.I),
             iota=np.ascontiguousarray(fld.iota))
    k.update(over.pop("arrays", {}))
    p = lambda a: a.ctypes.data_as(C.c_void_p)
    d = G.gc_field_desc(fld.ns, fld.nfp, fld.nh, p(k["xm"]), p(k["xn"]), p(k["bmnc"]), p(k["G"]), p(k["I"]),
                        p(k["iota"]), fld.psi0, 0, None, None, None, None, None)
    for name, v in over.items():
        setattr(d, name, v)
    return d, k


def test_argument_validation_needs_no_device(lib):
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld = W.make_field(0)
    h = C.c_void_p(None)
    assert lib.gc_field_create(None, C.byref(h)) == G.GC_EINVAL
    assert lib.gc_field_create(C.byref(_desc(fld)[0]), None) == G.GC_EINVAL
    for over in (dict(ns=3), dict(nfp=0), dict(nh=0), dict(nk=-1), dict(psi0=0.0), dict(xm=None), dict(nk=2)):
        d, keep = _desc(fld, **over)
        assert lib.gc_field_create(C.byref(d), C.byref(h)) == G.GC_EINVAL, over
        assert not h.value
        assert lib.gc_last_error() != b""
    bad = fld.bmnc.copy()
    bad[1, 1] = np.inf
    d, keep = _desc(fld, arrays=dict(bmnc=bad))
    assert lib.gc_field_create(C.byref(d), C.byref(h)) == G.GC_EINVAL
    assert b"non-finite" in lib.gc_last_error()
    assert lib.gc_field_destroy(None) == G.GC_OK
    assert lib.gc_trace(None, None, 0, *([None] * 15)) == G.GC_EINVAL
    assert lib.gc_trace_noalloc(None, None, 0, *([None] * 15)) == G.GC_EINVAL
    assert lib.gc_field_eval(None, 0, None, None, None, None, None, None) == G.GC_EINVAL


def test_no_cpu_fallback(lib):
    """Without a CUDA device a well-formed gc_field_create fails with GC_ECUDA; the Python binding raises."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld = W.make_field(0)
    d, keep = _desc(fld)
    h = C.c_void_p(None)
    assert lib.gc_field_create(C.byref(d), C.byref(h)) == G.GC_ECUDA
    assert b"no CPU fallback" in lib.gc_last_error()
    with pytest.raises(G.GcError):
        G.Field(fld)


def test_product_path_does_not_import_the_oracle():
    """Nothing under paper_2605_16734_b200/ or include/ names the oracle package or its library."""
    pkg = os.path.join(ROOT, "paper_2605_16734_b200")
    for base, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(base, f)).read()
                assert "import oracle" not in text and "libgc_oracle" not in text and "gc_oracle.h" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "gcorbit" not in text.replace("paper_2605_16734_b200/csrc", ""), f
