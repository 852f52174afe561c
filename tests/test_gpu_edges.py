"""-m gpu: edge cases of the boundary and of the controller (O6-O8), each against the oracle."""
from __future__ import annotations

import dataclasses

import numpy as np
import pytest

from gpu_common import assert_trace_parity, gpu_trace, make_case, rel_diff, sort_poincare, to_dev

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def case0():
    return make_case(0, 96)


@pytest.fixture(scope="module")
def case4():
    return make_case(4, 64)


def _kernels():
    from paper_2605_16734_b200 import gcorbit as G
    return [G.GC_KERNEL_GENERIC, G.GC_KERNEL_WARP, G.GC_KERNEL_TILE, G.GC_KERNEL_MMA]


def test_empty_ensemble(case0):
    import torch
    fld, spec, P, OF, GF, mu = case0
    e = torch.empty(0, dtype=torch.float64, device="cuda:0")
    r = GF.trace(spec, e, e, e, e, e)
    torch.cuda.synchronize()
    assert r.y.shape == (4, 0) and r.status.numel() == 0
    B, dB = GF.field_eval(e, e, e)
    assert B.numel() == 0


def test_t0_at_or_past_t_max_returns_inputs(case0):
    fld, spec, P, OF, GF, mu = case0
    for kern in _kernels():
        GF.set_kernel(kern)
        r = gpu_trace(GF, spec, P, mu, t0=1e-5, t_max=1e-5)
        assert (r.status.cpu().numpy() == 0).all()
        assert (r.n_acc.cpu().numpy() == 0).all() and (r.n_rej.cpu().numpy() == 0).all()
        y = r.y.cpu().numpy()
        assert np.array_equal(y[0], P.s) and np.array_equal(y[1], P.theta) and np.array_equal(y[2], P.zeta)
        assert np.abs(y[3] - P.vpar).max() <= 4e-16 * spec.v_ref          # v_par round-trips through u = v/v_ref
        assert (r.t.cpu().numpy() == 1e-5).all()


def test_start_outside_and_nonfinite(case0):
    """s0 >= s_loss is lost after its first accepted step; s0 <= s_min is an axis stop; NaN/inf inputs end
    with status 4 (O6, O7) -- the same on both sides."""
    fld, spec, P, OF, GF, mu = case0
    Q = P.head(8)
    Q.s[:] = [1.0, 1.05, 5e-4, 0.25, 0.25, 0.25, 0.25, 0.6]
    Q.theta[3] = np.nan
    Q.zeta[4] = np.inf
    m = mu[:8].copy()
    m[5] = np.nan
    o = OF.trace(spec, Q.s, Q.theta, Q.zeta, Q.vpar, m, t_max=2e-6)
    assert o.status[1] == 1 and o.status[2] == 2 and list(o.status[3:6]) == [4, 4, 4]
    for kern in _kernels():
        GF.set_kernel(kern)
        r = gpu_trace(GF, spec, Q, m, t_max=2e-6)
        assert np.array_equal(r.status.cpu().numpy(), o.status)
        ok = o.status != 4
        assert rel_diff(r.y.cpu().numpy()[:, ok], o.y[:, ok], spec.v_ref).max() < 1e-9
        assert np.array_equal(r.n_acc.cpu().numpy()[ok], o.n_acc[ok])


def test_max_steps_cap(case0):
    fld, spec, P, OF, GF, mu = case0
    sp = dataclasses.replace(spec, max_steps=7)
    o = OF.trace(sp, P.s, P.theta, P.zeta, P.vpar, mu)
    assert (o.status == 3).all()
    for kern in _kernels():
        GF.set_kernel(kern)
        r = gpu_trace(GF, sp, P, mu)
        assert (r.status.cpu().numpy() == 3).all()
        assert np.array_equal(r.n_acc.cpu().numpy() + r.n_rej.cpu().numpy(), np.full(P.n, 7))
        # A capped particle ends at ITS OWN time, not at a common t_max.  The first proposals h come from
        # err**-0.2 while the embedded error (|delta| ~ 1e-12 at h = 1e-8 s) still carries the rounding noise
        # of the harmonic sum at the 1e-6 level, so two correct implementations end ~1e-7 apart (relative)
        # in t and ydot * dt apart in y.  Compare after removing ydot * dt.
        same = (r.n_acc.cpu().numpy() == o.n_acc) & (r.n_rej.cpu().numpy() == o.n_rej)
        assert same.mean() >= 0.97
        yg, tg = r.y.cpu().numpy(), r.t.cpu().numpy()
        dt = tg - o.t
        assert (np.abs(dt) <= 1e-5 * o.t).all()
        floor = np.array([1.0, 1.0, 1.0, sp.v_ref])
        for i in np.nonzero(same)[0]:
            yo = o.y[:, i] / np.array([1.0, 1.0, 1.0, sp.v_ref])
            ydot = OF.rhs(sp.mass, sp.charge, mu[i], sp.v_ref, o.t[i], yo) * np.array([1.0, 1.0, 1.0, sp.v_ref])
            resid = np.abs(yg[:, i] - o.y[:, i] - ydot * dt[i]) / np.maximum(np.abs(o.y[:, i]), floor)
            assert resid.max() <= 1e-9, (i, resid)


def test_minimum_step_forces_acceptance(case0):
    """A9: with h_min above the natural step every attempt after a rejection is made at h_min and accepted
    whatever its error."""
    fld, spec, P, OF, GF, mu = case0
    sp = dataclasses.replace(spec, h_min=2e-7, h0=1e-6)
    o = OF.trace(sp, P.s, P.theta, P.zeta, P.vpar, mu, t_max=2e-5)
    assert o.n_forced.sum() > 0
    for kern in _kernels():
        GF.set_kernel(kern)
        r = gpu_trace(GF, sp, P, mu, t_max=2e-5)
        assert np.array_equal(r.status.cpu().numpy(), o.status)
        same = (r.n_acc.cpu().numpy() == o.n_acc) & (r.n_rej.cpu().numpy() == o.n_rej)
        assert same.mean() > 0.9
        assert np.array_equal(r.n_forced.cpu().numpy()[same], o.n_forced[same])
        # forced steps carry errors far above rtol: compare at the accuracy those steps have
        assert rel_diff(r.y.cpu().numpy()[:, same], o.y[:, same], sp.v_ref).max() < 1e-7


def test_forced_only_after_a_rejection_and_step_underflow(case0):
    """The three controller branches pinned on the oracle in tests/test_oracle_controller.py, on every kernel:
    h0 = h_min far above the natural step gives reject / forced accept pairs (5 + 5 with t_max = 4.5 h_min), never a
    forced first attempt; A23: t + h == t ends a particle with status 4 and zero attempts."""
    fld, spec, P, OF, GF, mu = case0
    Q = P.head(33)
    sp = dataclasses.replace(spec, h_min=4e-7, h0=4e-7)
    o = OF.trace(sp, Q.s, Q.theta, Q.zeta, Q.vpar, mu[:33], t_max=4.5 * 4e-7)
    assert (o.n_acc == 5).all() and (o.n_rej == 5).all() and (o.n_forced == 5).all()
    su = dataclasses.replace(spec, h_min=0.0, h0=1e-12, max_steps=1000)
    for kern in _kernels():
        GF.set_kernel(kern)
        r = gpu_trace(GF, sp, Q, mu[:33], t_max=4.5 * 4e-7)
        for a, b in ((r.n_acc, o.n_acc), (r.n_rej, o.n_rej), (r.n_forced, o.n_forced), (r.status, o.status)):
            assert np.array_equal(a.cpu().numpy(), b)
        assert (r.t.cpu().numpy() == 4.5 * 4e-7).all()
        assert rel_diff(r.y.cpu().numpy(), o.y, sp.v_ref).max() < 1e-7      # forced steps: far above rtol
        u = gpu_trace(GF, su, Q, mu[:33], t0=1e8, t_max=2e8)
        assert (u.status.cpu().numpy() == 4).all() and (u.t.cpu().numpy() == 1e8).all()
        assert (u.n_acc.cpu().numpy() == 0).all() and (u.n_rej.cpu().numpy() == 0).all()
        assert np.array_equal(u.y.cpu().numpy()[0], Q.s)
    GF.set_kernel(0)


def test_h_inout_roundtrip_and_segments(case0):
    """Two calls joined by h_inout and GC_TRACE_RESUME equal the oracle run with the same segmentation; lost
    or stopped particles are not touched by the second call."""
    import torch
    fld, spec, P, OF, GF, mu = case0
    Q = P.head(96)
    Q.s[:6] = 0.97                                                   # some of these are lost in segment 1
    t1, t2 = 1.5e-5, 3e-5
    o1 = OF.trace(spec, Q.s, Q.theta, Q.zeta, Q.vpar, mu, t0=0.0, t_max=t1)
    alive = o1.status == 0
    o2 = OF.trace(spec, o1.y[0, alive], o1.y[1, alive], o1.y[2, alive], o1.y[3, alive], mu[alive],
                  h_in=o1.h[alive], t0=t1, t_max=t2)
    for kern in _kernels():
        GF.set_kernel(kern)
        h = torch.zeros(Q.n, dtype=torch.float64, device="cuda:0")
        mu_d = to_dev(mu)
        st = GF.trace(spec, to_dev(Q.s), to_dev(Q.theta), to_dev(Q.zeta), to_dev(Q.vpar), mu_d, h_inout=h,
                      t0=0.0, t_max=t1)
        torch.cuda.synchronize()
        y1, s1 = st.y.cpu().numpy().copy(), st.status.cpu().numpy().copy()
        assert np.array_equal(s1, o1.status)
        # the proposal is h * 0.9 * err**-0.2 and err carries the rounding noise of the embedded error estimate
        dh = np.abs(h.cpu().numpy() / o1.h - 1)
        assert dh.max() < 1e-5 and np.median(dh) < 1e-8
        GF.trace_resume(spec, st, mu_d, t0=t1, t_max=t2)
        torch.cuda.synchronize()
        y2, s2 = st.y.cpu().numpy(), st.status.cpu().numpy()
        assert np.array_equal(y2[:, ~alive], y1[:, ~alive]) and np.array_equal(s2[~alive], s1[~alive])
        assert np.array_equal(s2[alive], o2.status)
        assert rel_diff(y2[:, alive], o2.y, spec.v_ref).max() < 1e-6
        assert np.median(rel_diff(y2[:, alive], o2.y, spec.v_ref)) < 1e-9
        # counters accumulate over the two calls
        tot = st.n_acc.cpu().numpy()[alive] + st.n_rej.cpu().numpy()[alive]
        ref = o1.n_acc[alive] + o1.n_rej[alive] + o2.n_acc + o2.n_rej
        assert (tot == ref).mean() > 0.97


def test_trace_host_equals_device_trace(case4):
    """gc_trace_host (host buffers, copies inside) returns bit-for-bit what gc_trace returns."""
    fld, spec, P, OF, GF, mu = case4
    r = gpu_trace(GF, spec, P, mu, t_max=1e-5, poincare_capacity=1024)
    hres = GF.trace_host(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=1e-5, poincare_capacity=1024)
    assert np.array_equal(hres.y, r.y.cpu().numpy())
    assert np.array_equal(hres.t, r.t.cpu().numpy())
    assert np.array_equal(hres.status, r.status.cpu().numpy())
    assert np.array_equal(hres.n_acc, r.n_acc.cpu().numpy())
    assert np.array_equal(hres.n_rej, r.n_rej.cpu().numpy())
    assert hres.poincare_count == r.poincare_count
    assert np.array_equal(sort_poincare(hres.poincare), sort_poincare(r.poincare.cpu().numpy()))


def test_poincare_overflow_keeps_counting(case4):
    fld, spec, P, OF, GF, mu = case4
    full = gpu_trace(GF, spec, P, mu, t_max=1e-5, poincare_capacity=4096)
    assert full.poincare_count > 8
    small = gpu_trace(GF, spec, P, mu, t_max=1e-5, poincare_capacity=8)
    assert small.poincare_count == full.poincare_count and small.poincare.shape[0] == 8
    # every kept record is one of the full run's records
    a = sort_poincare(full.poincare.cpu().numpy())
    for rec in small.poincare.cpu().numpy():
        assert (np.abs(a - rec).max(axis=1) == 0).any()


def test_invalid_arguments_are_reported(case0):
    import ctypes as C
    from paper_2605_16734_b200 import gcorbit as G
    fld, spec, P, OF, GF, mu = case0
    for bad in (dict(v_ref=0.0), dict(h0=0.0), dict(h_min=-1.0), dict(rtol=0.0, atol=0.0), dict(max_steps=0),
                dict(mass=0.0), dict(charge=0.0), dict(t_max=float("nan"))):
        with pytest.raises(G.GcError) as ei:
            gpu_trace(GF, dataclasses.replace(spec, **bad), P, mu)
        assert ei.value.code == G.GC_EINVAL, bad
    L = G.load_library()
    p = G.make_params(spec)
    assert L.gc_trace(GF._h, C.byref(p), 4, *([None] * 15)) == G.GC_EINVAL
    assert b"NULL" in L.gc_last_error()
    p.flags = 64
    assert L.gc_trace(GF._h, C.byref(p), 0, *([None] * 15)) == G.GC_EINVAL
    with pytest.raises(G.GcError):
        GF.set_kernel(99)


def test_field_create_rejects_bad_tables():
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld = W.make_field(0)
    bad = dataclasses.replace(fld, bmnc=fld.bmnc.copy())
    bad.bmnc[3, 5] = np.nan
    with pytest.raises(G.GcError) as ei:
        G.Field(bad)
    assert ei.value.code == G.GC_EINVAL
    bad = dataclasses.replace(fld, xm=-fld.xm)
    with pytest.raises(G.GcError):
        G.Field(bad)
    modes = W.make_field(2)
    bad = dataclasses.replace(modes, mode_omega=np.zeros_like(modes.mode_omega))
    with pytest.raises(G.GcError):
        G.Field(bad)
    small = dataclasses.replace(fld, ns=3, bmnc=fld.bmnc[:3], G=fld.G[:3], I=fld.I[:3], iota=fld.iota[:3])
    with pytest.raises(G.GcError):
        G.Field(small)


def test_fields_outside_the_warp_layout_use_the_generic_kernel():
    """max |xn| > 16 does not fit the packed layout: AUTO falls back to the generic kernel, which still
    matches the oracle; harmonics given in shuffled order with a duplicated (m, n) pair add up."""
    import oracle
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld = W.make_equilibrium(4, 20, 31)
    GF = G.Field(fld)
    assert GF.kernel_info()["kernel"] == "generic"
    with pytest.raises(G.GcError):
        GF.set_kernel(G.GC_KERNEL_WARP)
    spec = W.make_spec(0)
    P = W.make_particles(0, 40)
    OF = oracle.OracleField(fld)
    mu = W.mu_from(P, OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    r = gpu_trace(GF, spec, P, mu, t_max=5e-6)
    o = OF.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=5e-6)
    assert_trace_parity(r, o, spec, min_same=0.95, label="generic N=20")

    base = W.make_field(0)
    perm = np.random.default_rng(3).permutation(base.nh)
    xm = np.concatenate([base.xm[perm], base.xm[10:11]])
    xn = np.concatenate([base.xn[perm], base.xn[10:11]])
    bm = np.concatenate([base.bmnc[:, perm], 0.5 * base.bmnc[:, 10:11]], axis=1)
    shuf = dataclasses.replace(base, xm=xm, xn=xn, bmnc=np.ascontiguousarray(bm))
    GF2, OF2 = G.Field(shuf), oracle.OracleField(shuf)
    assert GF2.kernel_info(40)["kernel"] == "warp" and GF2.kernel_info(100_000)["kernel"] == "mma"
    mu2 = W.mu_from(P, OF2.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    r = gpu_trace(GF2, spec, P, mu2, t_max=5e-6)
    o = OF2.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu2, t_max=5e-6)
    assert_trace_parity(r, o, spec, min_same=0.95, label="shuffled harmonics")


@pytest.mark.parametrize("kernel", ["tile", "mma"])
def test_binned_kernels_are_bitwise_reproducible_and_independent_of_the_company(kernel):
    """The binned kernels scatter particles with atomics, so which particles share a tile / a DMMA group differs from
    run to run and with the ensemble around them.  A particle's result must not depend on it (rows
    outside a particle's stencil carry weight exactly 0; window and global-memory sweeps use one instruction
    sequence): two runs of 30,000 particles agree bit for bit, and so do the first 5,000 particles traced alone
    (other tiles, other groups, smaller tiles)."""
    import torch
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld, spec = W.make_field(4), W.make_spec(4)
    P = W.make_particles(4, 30_000)
    GF = G.Field(fld)
    GF.set_kernel({"tile": G.GC_KERNEL_TILE, "mma": G.GC_KERNEL_MMA}[kernel])
    s, th, ze, vp = (to_dev(x) for x in (P.s, P.theta, P.zeta, P.vpar))
    B, _ = GF.field_eval(s, th, ze, derivs=False)
    mu = to_dev(0.5 * spec.mass * P.vperp2()) / B
    run = lambda k: GF.trace(spec, s[:k].contiguous(), th[:k].contiguous(), ze[:k].contiguous(),
                             vp[:k].contiguous(), mu[:k].contiguous(), t_max=3e-6)
    a, b, c = run(P.n), run(P.n), run(5000)
    torch.cuda.synchronize()
    for x, y in ((a, b), ):
        assert torch.equal(x.y, y.y) and torch.equal(x.t, y.t) and torch.equal(x.status, y.status)
        assert torch.equal(x.n_acc, y.n_acc) and torch.equal(x.n_rej, y.n_rej)
    assert torch.equal(a.y[:, :5000], c.y) and torch.equal(a.t[:5000], c.t) and torch.equal(a.n_acc[:5000], c.n_acc)


@pytest.mark.parametrize("kernel", ["tile", "mma"])
def test_streaming_through_few_record_slots_changes_nothing(kernel):
    """GC_OPT_WAVE_PARTICLES: 30,000 particles streamed through 4096 record slots (a finished particle hands its slot
    to the next unstarted one) give bit for bit the results of one slot per particle -- also for a resumed second
    segment in which lost particles are passed over, with samples, and for the right-hand side alone."""
    import torch
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld, spec = W.make_field(1), W.make_spec(1)
    P = W.make_particles(1, 30_000)
    P.s[::7] = 0.97 + 0.02 * P.s[::7]                       # a good share of early losses (uneven slot turnover)
    GF = G.Field(fld)
    GF.set_kernel({"tile": G.GC_KERNEL_TILE, "mma": G.GC_KERNEL_MMA}[kernel])
    s, th, ze, vp = (to_dev(x) for x in (P.s, P.theta, P.zeta, P.vpar))
    B, _ = GF.field_eval(s, th, ze, derivs=False)
    mu = to_dev(0.5 * spec.mass * P.vperp2()) / B

    def two_segments():
        h = torch.zeros(P.n, dtype=torch.float64, device="cuda:0")
        st = GF.trace(spec, s, th, ze, vp, mu, h_inout=h, t0=0.0, t_max=4e-6)
        first = (st.y.clone(), st.t.clone(), st.status.clone(), st.n_acc.clone())
        GF.trace_resume(spec, st, mu, t0=4e-6, t_max=6e-6)
        smp = GF.trace_sampled(spec, s, th, ze, vp, mu, 0.0, 1e-6, 4, t_max=3e-6)
        y4 = torch.stack([s, th, ze, vp]).contiguous()
        rhs = GF.rhs_eval(spec.mass, spec.charge, 0.0, y4, mu)
        torch.cuda.synchronize()
        return first, st, smp, rhs

    f0, a, sa, ra = two_segments()
    GF.set_option(G.GC_OPT_WAVE_PARTICLES, 4096)
    f1, b, sb, rb = two_segments()
    GF.set_option(G.GC_OPT_WAVE_PARTICLES, 0)
    lost = int((f0[2] == 1).sum())
    assert 1000 < lost < 20_000                             # the resumed call really passes particles over
    for x, y in zip(f0, f1):
        assert torch.equal(x, y)
    for name in ("y", "t", "status", "n_acc", "n_rej", "n_forced", "h"):
        assert torch.equal(getattr(a, name), getattr(b, name)), name
    assert torch.equal(sa.sample_end, sb.sample_end)
    assert torch.equal(torch.nan_to_num(sa.samples, nan=-7.0), torch.nan_to_num(sb.samples, nan=-7.0))
    assert torch.equal(ra, rb)
    with pytest.raises(G.GcError):
        GF.set_option(G.GC_OPT_WAVE_PARTICLES, 100)
    with pytest.raises(G.GcError):
        GF.set_option(77, 1)


@pytest.mark.parametrize("kernel", ["generic", "warp", "tile", "mma"])
def test_refined_loss_point_matches_oracle(kernel):
    """GC_TRACE_REFINE_LOSS (O7b): lost particles report the crossing of s_loss on the continuous extension; the
    warp kernel hands the call to the generic one.  Everything else equals the unrefined trace."""
    import dataclasses
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    fld, spec, P, OF, GF, mu = make_case(0, 96)
    spec = dataclasses.replace(spec, s_loss=0.262)
    GF.set_kernel({"generic": G.GC_KERNEL_GENERIC, "warp": G.GC_KERNEL_WARP, "tile": G.GC_KERNEL_TILE,
                   "mma": G.GC_KERNEL_MMA}[kernel])
    a = [to_dev(x) for x in (P.s, P.theta, P.zeta, P.vpar, mu)]
    r = GF.trace(spec, *a, t_max=3e-5, flags=G.GC_TRACE_REFINE_LOSS)
    u = GF.trace(spec, *a, t_max=3e-5)
    torch.cuda.synchronize()
    o = OF.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=3e-5, refine_loss=True)
    st = r.status.cpu().numpy()
    assert np.array_equal(st, o.status) and 10 < (st == 1).sum() < 90
    same = (r.n_acc.cpu().numpy() == o.n_acc) & (r.n_rej.cpu().numpy() == o.n_rej)
    assert same.mean() >= 0.97
    lost = (st == 1) & same
    y, t = r.y.cpu().numpy(), r.t.cpu().numpy()
    assert np.abs(y[0, lost] - spec.s_loss).max() < 1e-12
    assert np.abs(t[lost] - o.t[lost]).max() <= 1e-9 * 3e-5
    floor = np.array([[1.0], [1.0], [1.0], [spec.v_ref]])
    assert (np.abs(y[:, lost] - o.y[:, lost]) / np.maximum(np.abs(o.y[:, lost]), floor)).max() < 1e-9
    # refined times precede the step ends of the unrefined trace by less than a step; survivors are identical
    tu = u.t.cpu().numpy()
    assert np.all(t[lost] <= tu[lost]) and np.all(tu[lost] - t[lost] < 2e-7)
    surv = torch.as_tensor(st == 0)
    if kernel == "warp":                                   # the refined call ran in the generic kernel: rounding differs
        d = (r.y[:, surv] - u.y[:, surv]).abs() / torch.maximum(u.y[:, surv].abs(), to_dev(floor))
        assert float(d.max()) < 1e-9
    else:
        assert torch.equal(r.y[:, surv], u.y[:, surv]) and torch.equal(r.n_acc, u.n_acc)


def test_two_live_fields_sharing_a_kernel_instantiation():
    """The dynamic shared-memory limit belongs to the kernel function, not to a field: a field with a large window
    (config 4, 16 mode harmonics) must still launch after a field with a smaller window of the same instantiation
    (config 2, 8 mode harmonics) was created."""
    from paper_2605_16734_b200 import gcorbit as G
    fld4, spec4, P4, OF4, GF4, mu4 = make_case(4, 4200)
    fld2, spec2, P2, OF2, GF2, mu2 = make_case(2, 64)          # created second: used to lower the limit
    k = 24
    o = OF4.trace(spec4, P4.s[:k], P4.theta[:k], P4.zeta[:k], P4.vpar[:k], mu4[:k], t_max=2e-6)
    for kern in (G.GC_KERNEL_TILE, G.GC_KERNEL_MMA):
        GF4.set_kernel(kern)
        r = gpu_trace(GF4, spec4, P4, mu4, t_max=2e-6)
        assert np.array_equal(r.status.cpu().numpy()[:k], o.status)
        assert rel_diff(r.y.cpu().numpy()[:, :k], o.y, spec4.v_ref).max() < 1e-9
        GF2.set_kernel(kern)
        r2 = gpu_trace(GF2, spec2, P2, mu2, t_max=1e-6)
        assert (r2.status.cpu().numpy() == 0).all()


def test_trace_host_refuses_overlapping_calls_on_one_field(case0):
    """gc_trace_host keeps its device workspace in the field, so it is not re-entrant on one field: a call that
    overlaps another one returns GC_EINVAL instead of corrupting the workspace (include/gcorbit.h)."""
    import threading
    from paper_2605_16734_b200 import gcorbit as G
    fld, spec, P, OF, GF, mu = case0
    GF.set_kernel(G.GC_KERNEL_GENERIC)                         # slow on purpose: the first call runs for a while
    results = []

    def call(t_max):
        try:
            r = GF.trace_host(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=t_max)
            results.append(("ok", r))
        except G.GcError as e:
            results.append(("err", e))

    a = threading.Thread(target=call, args=(5e-4,))
    a.start()
    import time
    time.sleep(0.05)
    call(1e-6)                                                 # overlaps the first call (ctypes releases the GIL)
    a.join()
    GF.set_kernel(G.GC_KERNEL_AUTO)
    kinds = sorted(k for k, _ in results)
    assert kinds == ["err", "ok"], kinds
    err = [v for k, v in results if k == "err"][0]
    assert err.code == G.GC_EINVAL and "another gc_trace_host call" in str(err)
    again = GF.trace_host(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=1e-6)      # and the field is usable afterwards
    assert (again.status == 0).all()


def test_chunk_option_beyond_the_compiled_maximum_is_refused(case0):
    """GC_OPT_CHUNK_ATTEMPTS: gcorbit.h promises GC_EINVAL for a value out of range; the kernels are compiled for at
    most 8 attempted steps per chunk, and a larger value used to be clamped silently."""
    from paper_2605_16734_b200 import gcorbit as G
    fld, spec, P, OF, GF, mu = case0
    for ok in (0, 1, 8):
        GF.set_option(G.GC_OPT_CHUNK_ATTEMPTS, ok)
    for bad in (9, 64, 1000):
        with pytest.raises(G.GcError) as e:
            GF.set_option(G.GC_OPT_CHUNK_ATTEMPTS, bad)
        assert e.value.code == G.GC_EINVAL
    GF.set_option(G.GC_OPT_CHUNK_ATTEMPTS, 0)

