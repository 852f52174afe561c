"""-m gpu: gc_trace_noalloc against gc_trace.

gc_trace_noalloc exists for programs that embed libgcorbit.so but are not allowed to allocate GPU memory while they
run: a service whose own arena took the whole device at start-up, a loop with a deadline that cannot absorb the
stalls of the driver's allocator, a plug-in whose host owns every allocation.  It is the mma trace kernel with its
work area in a fixed 5 MiB array inside the library image instead of pool memory, so its results must be those of
gc_trace with GC_KERNEL_MMA.  Every call shares that one array and finds in it what the call before left, hence the
test makes two calls in a row, the second one smaller, on another field (another carve-up of the array) and with
Poincare records, and compares each with the existing path; it also checks that an ensemble beyond the fixed size is
refused with an error that names the limit.

The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It passes alone in a fresh process (then its first call also does the per-GPU set-up) and after the others.
"""
from __future__ import annotations

import numpy as np
import pytest

from gpu_common import SAME_RTOL, rel_diff, sort_poincare, to_dev

pytestmark = pytest.mark.gpu


def _ensemble(config, n):
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    GF = G.Field(W.make_field(config))
    spec = W.make_spec(config)
    P = W.make_particles(config, n)
    s, th, ze, vp = (to_dev(x) for x in (P.s, P.theta, P.zeta, P.vpar))
    B, _ = GF.field_eval(s, th, ze, derivs=False)
    mu = to_dev(0.5 * spec.mass * P.vperp2()) / B
    return GF, spec, (s, th, ze, vp, mu)


def _buffers(n, capacity=0):
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    i32 = lambda: torch.full((n,), -7, dtype=torch.int32, device="cuda:0")
    out = G.TraceResult(torch.full((4, n), np.nan, dtype=torch.float64, device="cuda:0"),
                        torch.full((n,), np.nan, dtype=torch.float64, device="cuda:0"), i32(), i32(), i32(), i32(), None)
    if capacity:
        out.poincare = torch.zeros((capacity, 4), dtype=torch.float64, device="cuda:0")
    return out


def _assert_same(new, old, spec, label):
    """The tolerance of the parity tests (flat 1e-9 on the states and the end time, identical status and attempt
    counters); the two launches differ only in where the work area lives, so they are expected to agree exactly."""
    for name in ("status", "n_acc", "n_rej", "n_forced"):
        a, b = getattr(new, name).cpu().numpy(), getattr(old, name).cpu().numpy()
        assert np.array_equal(a, b), f"{label}: {name} differs at {np.nonzero(a != b)[0][:8]}"
    yn, yo = new.y.cpu().numpy(), old.y.cpu().numpy()
    assert np.isfinite(yn).all(), f"{label}: an output row was left unwritten"
    assert rel_diff(yn, yo, spec.v_ref).max() <= SAME_RTOL, label
    tn, to = new.t.cpu().numpy(), old.t.cpu().numpy()
    assert (np.abs(tn - to) <= SAME_RTOL * np.maximum(np.abs(to), 1e-300)).all(), label
    hn, ho = new.h.cpu().numpy(), old.h.cpu().numpy()
    assert (np.abs(hn - ho) <= SAME_RTOL * np.abs(ho)).all(), label


def test_noalloc_trace_matches_gc_trace_on_two_calls_in_a_row():
    import torch
    from paper_2605_16734_b200 import gcorbit as G

    # call 1: config 1 (101 radial nodes), 6001 particles = several tiles per cell and a ragged last one
    GF1, spec1, in1 = _ensemble(1, 6001)
    h_new = torch.zeros(6001, dtype=torch.float64, device="cuda:0")
    new1 = GF1.trace_noalloc(spec1, *in1, out=_buffers(6001), h_inout=h_new, t_max=2e-5)
    # call 2, straight after it on the same stream: another field (51 nodes: the index arrays land elsewhere in the
    # array, on top of what call 1 left), fewer particles, Poincare records
    cap = 1 << 16
    GF0, spec0, in0 = _ensemble(0, 1187)
    h_new0 = torch.zeros(1187, dtype=torch.float64, device="cuda:0")
    count = torch.full((1,), 12345, dtype=torch.int64, device="cuda:0")
    new0 = GF0.trace_noalloc(spec0, *in0, out=_buffers(1187, cap), h_inout=h_new0, t_max=2e-5, poincare_count=count)
    torch.cuda.synchronize()
    G.finish_poincare(new0)

    # the existing path: gc_trace on the mma kernel, pool memory
    for GF in (GF1, GF0):
        GF.set_kernel(G.GC_KERNEL_MMA)
    h_old = torch.zeros(6001, dtype=torch.float64, device="cuda:0")
    old1 = GF1.trace(spec1, *in1, h_inout=h_old, t_max=2e-5)
    h_old0 = torch.zeros(1187, dtype=torch.float64, device="cuda:0")
    old0 = GF0.trace(spec0, *in0, h_inout=h_old0, t_max=2e-5, poincare_capacity=cap)
    torch.cuda.synchronize()
    G.finish_poincare(old0)

    assert (new1.status.cpu().numpy() >= 0).all() and (new1.n_acc.cpu().numpy() > 0).all()
    _assert_same(new1, old1, spec1, "call 1 (config 1, 6001 particles)")
    _assert_same(new0, old0, spec0, "call 2 (config 0, 1187 particles)")
    assert 0 < new0.poincare_count == old0.poincare_count <= cap
    rn, ro = sort_poincare(new0.poincare.cpu().numpy()), sort_poincare(old0.poincare.cpu().numpy())
    assert np.array_equal(rn[:, 0], ro[:, 0])
    assert np.abs(rn[:, 1:] - ro[:, 1:]).max() <= SAME_RTOL * np.maximum(np.abs(ro[:, 1:]), 1.0).max()

    # a third call reusing call 1's buffers gives call 1's result again (the array carries nothing over)
    again = GF1.trace_noalloc(spec1, *in1, out=_buffers(6001), h_inout=torch.zeros_like(h_new), t_max=2e-5)
    torch.cuda.synchronize()
    assert torch.equal(again.y, new1.y) and torch.equal(again.status, new1.status)
    GF1.close(); GF0.close()


def test_noalloc_refuses_what_does_not_fit():
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    n = G.NOALLOC_MAX_PARTICLES + 1
    GF, spec, inp = _ensemble(0, n)
    with pytest.raises(G.GcError) as e:
        GF.trace_noalloc(spec, *inp, out=_buffers(n), t_max=1e-6)
    assert e.value.code == G.GC_EINVAL and "GC_NOALLOC_MAX_PARTICLES" in str(e.value)
    # the largest ensemble that fits runs, on a field with many radial nodes too
    m = G.NOALLOC_MAX_PARTICLES
    r = GF.trace_noalloc(spec, *(x[:m].contiguous() for x in inp), out=_buffers(m), t_max=1e-6)
    GF.set_kernel(G.GC_KERNEL_MMA)
    o = GF.trace(spec, *(x[:m].contiguous() for x in inp), t_max=1e-6)
    torch.cuda.synchronize()
    assert torch.equal(r.status, o.status) and rel_diff(r.y.cpu().numpy(), o.y.cpu().numpy(), spec.v_ref).max() <= SAME_RTOL
    # a field with a 3-D interpolant is traced by another kernel: refused, not silently run on the direct sum
    GF.set_kernel(G.GC_KERNEL_AUTO)
    GF.set_grid(16, 16, 16, G.GC_GRID_HERMITE)
    with pytest.raises(G.GcError):
        GF.trace_noalloc(spec, *(x[:64].contiguous() for x in inp), out=_buffers(64), t_max=1e-6)
    GF.close()
