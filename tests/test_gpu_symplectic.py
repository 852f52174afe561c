"""-m gpu: NEXT-3 of SURVEY.md section 8(f) on the device -- gc_trace_symplectic (kernels_symplectic.cuh) against the
oracle's symplectic explicit-implicit Euler integrator (reading A28), element by element through
the C ABI, on the direct harmonic sum and on the 3-D interpolant (NEXT-2).

Both sides solve the same 2 x 2 system per step to a last update below 1e-13 (the oracle by Newton with a
finite-difference Jacobian, the device by a quasi-Newton iteration that needs one field evaluation per iteration), so
per step they agree to ~1e-13 and over N steps of a regular orbit to ~N x 1e-13 times the orbit's own error growth;
the bound is north_star's relative 1e-9 over short horizons."""
from __future__ import annotations

import numpy as np
import pytest

from gpu_common import make_case, record_info, rel_diff, to_dev

pytestmark = pytest.mark.gpu


def _chi(fld):
    s = np.arange(fld.ns) / (fld.ns - 1)
    return fld.psi0 * (0.42 * s + 0.05 * s ** 2)            # iota = 0.42 + 0.1 s of the BASELINE recipes


def _run_both(fld, spec, P, OF, GF, mu, dt, nsteps, **kw):
    import torch
    chi = _chi(fld)
    r = GF.trace_symplectic(spec.mass, spec.charge, to_dev(P.s), to_dev(P.theta), to_dev(P.zeta), to_dev(P.vpar),
                            to_dev(mu), to_dev(chi), dt, nsteps, **kw)
    torch.cuda.synchronize()
    o = OF.trace_symplectic(spec.mass, spec.charge, P.s, P.theta, P.zeta, P.vpar, mu, chi, dt, nsteps,
                            **{k: v for k, v in kw.items() if k != "max_iter"})
    return r, o


@pytest.mark.parametrize("grid", [None, ("lagrange", (51, 40, 36)), ("hermite", (51, 40, 36))])
@pytest.mark.parametrize("config,n,dt,nsteps", [(0, 300, 1e-8, 600), (1, 200, 2e-8, 250), (3, 257, 4e-8, 150)])
def test_symplectic_trace_matches_oracle(config, n, dt, nsteps, grid):
    fld, spec, P, OF, GF, mu = make_case(config, n)
    if grid:
        from paper_2605_16734_b200 import gcorbit as G, workloads as W
        if grid[0] == "hermite":
            OF.set_grid_hermite(*grid[1])
            GF.set_grid(*grid[1], kind=G.GC_GRID_HERMITE)
        else:
            OF.set_grid(*grid[1])
            GF.set_grid(*grid[1])
        mu = W.mu_from(P, OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    r, o = _run_both(fld, spec, P, OF, GF, mu, dt, nsteps)
    assert np.array_equal(r.status.cpu().numpy(), o.status)
    assert np.array_equal(r.n_steps.cpu().numpy(), o.n_steps)
    assert np.allclose(r.t.cpu().numpy(), o.t, rtol=1e-15, atol=0)
    ok = o.status != 4
    rel = rel_diff(r.y.cpu().numpy()[:, ok], o.y[:, ok], spec.v_ref)
    it = r.n_iter.cpu().numpy() / np.maximum(o.n_steps, 1)
    record_info("symplectic_parity", label=f"config {config} {grid[0] + ' grid' if grid else 'sum'} dt={dt:g} x {nsteps}",
                particles=int(ok.sum()), max_rel=float(rel.max()), median_rel=float(np.median(rel)),
                iterations_per_step=float(it.mean()), oracle_iterations_per_step=float((o.n_iter / np.maximum(o.n_steps, 1)).mean()))
    assert rel.max() < 1e-9 and np.median(rel) < 1e-11, (rel.max(), np.median(rel))
    assert 2.0 <= it.mean() <= 12.0


def test_symplectic_stop_rules_samples_resume_and_errors():
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    fld, spec, P, OF, GF, mu = make_case(0, 64)
    # loss / axis surfaces close to the start radius, samples every 100 steps
    kw = dict(t0=1e-6, s_loss=0.2502, s_min=0.2498, sample_stride=100, nsamp=7)
    r, o = _run_both(fld, spec, P, OF, GF, mu, 5e-9, 600, **kw)
    st = r.status.cpu().numpy()
    assert np.array_equal(st, o.status) and (st == 1).any() and (st == 2).any()
    assert np.array_equal(r.n_steps.cpu().numpy(), o.n_steps)
    assert np.array_equal(r.sample_end.cpu().numpy(), o.sample_end)
    assert np.allclose(r.t.cpu().numpy(), o.t, rtol=1e-15, atol=0)
    assert rel_diff(r.y.cpu().numpy(), o.y, spec.v_ref).max() < 1e-10
    S, So = r.samples.cpu().numpy(), o.samples
    valid = np.arange(7)[:, None] < o.sample_end[None, :]
    floor = np.array([1.0, 1.0, 1.0, spec.v_ref])[:, None, None]
    d = np.abs(S - So) / np.maximum(np.abs(So), floor)
    assert d[:, valid].max() < 1e-10
    assert np.isnan(S[:, ~valid]).all()                      # untouched
    # two resumed halves == one call (fixed step: the same map applied 600 times), bit for bit
    chi = to_dev(_chi(fld))
    a = [to_dev(x) for x in (P.s, P.theta, P.zeta, P.vpar, mu)]
    one = GF.trace_symplectic(spec.mass, spec.charge, *a, chi, 5e-9, 600)
    two = GF.trace_symplectic(spec.mass, spec.charge, *a, chi, 5e-9, 300)
    y = two.y
    GF.trace_symplectic(spec.mass, spec.charge, y[0], y[1], y[2], y[3], a[4], chi, 5e-9, 300, t0=300 * 5e-9, out=two,
                        flags=G.GC_TRACE_RESUME)
    torch.cuda.synchronize()
    assert np.array_equal(two.n_steps.cpu().numpy(), one.n_steps.cpu().numpy())
    # v_par -> p_zeta -> v_par at the hand-over costs rounding only
    assert rel_diff(two.y.cpu().numpy(), one.y.cpu().numpy(), spec.v_ref).max() < 1e-12
    # non-finite start -> status 4 without steps; empty ensemble; bad arguments; fields with modes are refused
    bad = [to_dev(np.array(v)) for v in ([np.nan], [0.0], [0.0], [1e6], [1e-14])]
    b = GF.trace_symplectic(spec.mass, spec.charge, *bad, chi, 5e-9, 5)
    torch.cuda.synchronize()
    assert int(b.status[0]) == 4 and int(b.n_steps[0]) == 0
    e = [to_dev(np.zeros(0)) for _ in range(5)]
    assert GF.trace_symplectic(spec.mass, spec.charge, *e, chi, 5e-9, 5).y.shape == (4, 0)
    for kwbad in (dict(dt=-1.0), dict(newton_tol=0.0), dict(max_iter=0)):
        args = dict(dt=5e-9, nsteps=5)
        args.update(kwbad)
        with pytest.raises(G.GcError) as ei:
            GF.trace_symplectic(spec.mass, spec.charge, *a, chi, args.pop("dt"), args.pop("nsteps"), **args)
        assert ei.value.code == G.GC_EINVAL
    fld2, spec2, P2, OF2, GF2, mu2 = make_case(2, 8)
    with pytest.raises(G.GcError):
        GF2.trace_symplectic(spec2.mass, spec2.charge, *[to_dev(x) for x in (P2.s, P2.theta, P2.zeta, P2.vpar, mu2)],
                             to_dev(_chi(fld2)), 5e-9, 5)


def test_symplectic_energy_is_bounded_while_dormand_prince_drifts_on_the_device():
    """PAPER.md:60-62 / Fig. 1 left with the device on both sides: gc_trace_symplectic against gc_trace_sampled at a
    loose tolerance, smooth field (cubic-in-s amplitudes), 4e-4 s."""
    import torch
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    import oracle
    fld = W.make_field(0)
    s = np.arange(fld.ns) / (fld.ns - 1)
    amp = fld.bmnc[-1, :].copy()
    fld.bmnc = np.ascontiguousarray(amp[None, :] * (0.2 * s + 0.8 * s ** 2 - 0.3 * s ** 3)[:, None])
    fld.bmnc[:, 0] = W.B00
    spec = W.make_spec(0)
    P = W.make_particles(0).head(32)
    GF = G.Field(fld)
    a = [to_dev(x) for x in (P.s, P.theta, P.zeta, P.vpar)]
    B0, _ = GF.field_eval(a[0], a[1], a[2], derivs=False)
    mu = to_dev(0.5 * spec.mass * P.vperp2()) / B0
    dt, nsteps, stride = 2.5e-8, 16000, 20
    nsamp = nsteps // stride + 1
    r = GF.trace_symplectic(spec.mass, spec.charge, *a, mu, to_dev(_chi(fld)), dt, nsteps, sample_stride=stride,
                            nsamp=nsamp)
    spec.rtol = spec.atol = 1e-6
    d = GF.trace_sampled(spec, *a, mu, 0.0, dt * stride, nsamp, t_max=dt * nsteps)
    torch.cuda.synchronize()
    keep = ((r.status == 0) & (d.status == 0)).cpu().numpy()              # a few of the 32 leave through s = 1
    assert keep.sum() >= 24 and (r.sample_end.cpu().numpy()[keep] == nsamp).all()

    def energy(S):
        Bs, _ = GF.field_eval(S[0].reshape(-1), S[1].reshape(-1), S[2].reshape(-1), derivs=False)
        return 0.5 * spec.mass * S[3] ** 2 + mu[None, :] * Bs.reshape(S[0].shape)
    Es, Ed = energy(r.samples).cpu().numpy(), energy(d.samples).cpu().numpy()
    es, ed = (Es / Es[0] - 1.0)[:, keep], (Ed / Ed[0] - 1.0)[:, keep]
    w = nsamp // 4
    drift_s = np.abs(es[-w:].mean(axis=0) - es[:w].mean(axis=0))
    drift_d = np.abs(ed[-w:].mean(axis=0) - ed[:w].mean(axis=0))
    amp_s = es.max(axis=0) - es.min(axis=0)
    assert amp_s.max() < 3e-2
    assert (drift_s < 0.02 * amp_s).all()
    assert np.median(drift_d) > 5 * np.median(drift_s)
    record_info("symplectic_energy", label=f"config-0 smooth field, {int(keep.sum())} particles, 4e-4 s",
                sym_amp_max=float(amp_s.max()), sym_drift_median=float(np.median(drift_s)),
                dp5_rtol1e6_drift_median=float(np.median(drift_d)))


@pytest.mark.parametrize("config,n,dt,nsteps", [(0, 2048 + 37, 1e-8, 300), (1, 3072 + 5, 2e-8, 100)])
def test_symplectic_on_the_mma_engine_matches_oracle_and_the_lane_kernel(config, n, dt, nsteps):
    """Ensembles of at least GC_TILE_MIN_PARTICLES(_SMALL) on the direct sum run through the cell-binned mma engine
    (trace_mma_symplectic_kernel: one pass of a lane = one field evaluation = one quasi-Newton iteration); smaller ones
    and GC_KERNEL_GENERIC through the lane kernel.  Both against the oracle, with stop surfaces close enough that all
    three exits occur."""
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    fld, spec, P, OF, GF, mu = make_case(config, n)
    lo, hi = float(np.quantile(P.s, 0.02)), float(np.quantile(P.s, 0.98))
    kw = dict(s_loss=hi + 2e-4, s_min=max(lo - 2e-4, 1e-3))
    if config == 0:                                          # every particle starts on s = 0.25
        kw = dict(s_loss=0.2515, s_min=0.2485)
    r, o = _run_both(fld, spec, P, OF, GF, mu, dt, nsteps, **kw)
    GF.set_kernel(G.GC_KERNEL_GENERIC)
    g = GF.trace_symplectic(spec.mass, spec.charge, to_dev(P.s), to_dev(P.theta), to_dev(P.zeta), to_dev(P.vpar),
                            to_dev(mu), to_dev(_chi(fld)), dt, nsteps, **kw)
    GF.set_kernel(G.GC_KERNEL_AUTO)
    torch.cuda.synchronize()
    st = r.status.cpu().numpy()
    assert np.array_equal(st, o.status) and np.array_equal(g.status.cpu().numpy(), o.status)
    assert (st == 0).any() and ((st == 1).any() or (st == 2).any())
    assert np.array_equal(r.n_steps.cpu().numpy(), o.n_steps) and np.array_equal(g.n_steps.cpu().numpy(), o.n_steps)
    assert np.allclose(r.t.cpu().numpy(), o.t, rtol=1e-15, atol=0)
    rel = rel_diff(r.y.cpu().numpy(), o.y, spec.v_ref)
    relg = rel_diff(g.y.cpu().numpy(), o.y, spec.v_ref)
    it = r.n_iter.cpu().numpy().sum() / max(o.n_steps.sum(), 1)
    record_info("symplectic_parity", label=f"config {config} sum, mma engine, {n} particles dt={dt:g} x {nsteps}",
                particles=n, max_rel=float(rel.max()), median_rel=float(np.median(rel)), iterations_per_step=float(it),
                oracle_iterations_per_step=float(o.n_iter.sum() / max(o.n_steps.sum(), 1)))
    assert rel.max() < 1e-9 and np.median(rel) < 1e-11, (rel.max(), np.median(rel))
    assert relg.max() < 1e-9
    # the two device paths iterate alike (the final pass of the binned path counts as one more evaluation per particle)
    assert abs(it - g.n_iter.cpu().numpy().sum() / max(o.n_steps.sum(), 1)) < 0.1
    # two resumed halves on the mma engine against one call
    a = [to_dev(x) for x in (P.s, P.theta, P.zeta, P.vpar, mu)]
    chi = to_dev(_chi(fld))
    h = nsteps // 2
    two = GF.trace_symplectic(spec.mass, spec.charge, *a, chi, dt, h, **kw)
    y = two.y
    GF.trace_symplectic(spec.mass, spec.charge, y[0], y[1], y[2], y[3], a[4], chi, dt, nsteps - h, t0=h * dt, out=two,
                        flags=G.GC_TRACE_RESUME, **kw)
    torch.cuda.synchronize()
    assert np.array_equal(two.status.cpu().numpy(), o.status)
    assert np.array_equal(two.n_steps.cpu().numpy(), o.n_steps)
    assert rel_diff(two.y.cpu().numpy(), o.y, spec.v_ref).max() < 1e-9


def test_symplectic_mma_engine_streams_through_few_record_slots():
    """The streaming case of the mma symplectic engine: 4096 record slots (GC_OPT_WAVE_PARTICLES) for 20 011 particles,
    so that slots are handed from finished particles to waiting ones inside one launch, in two resumed halves.  The
    result must not depend on the number of slots (bit for bit against one slot per particle) and a sample of the
    particles is checked against the oracle."""
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    n, dt, nsteps = 20011, 2e-8, 60
    fld, spec, P, OF, GF, mu = make_case(1, n)
    lo, hi = float(np.quantile(P.s, 0.02)), float(np.quantile(P.s, 0.98))
    kw = dict(s_loss=hi + 2e-4, s_min=max(lo - 2e-4, 1e-3))
    a = [to_dev(x) for x in (P.s, P.theta, P.zeta, P.vpar, mu)]
    chi = to_dev(_chi(fld))
    one = GF.trace_symplectic(spec.mass, spec.charge, *a, chi, dt, nsteps, **kw)       # a slot per particle, one call
    GF.set_option(G.GC_OPT_WAVE_PARTICLES, 4096)
    h = nsteps // 2
    two = GF.trace_symplectic(spec.mass, spec.charge, *a, chi, dt, h, **kw)
    y = two.y
    GF.trace_symplectic(spec.mass, spec.charge, y[0], y[1], y[2], y[3], a[4], chi, dt, nsteps - h, t0=h * dt, out=two,
                        flags=G.GC_TRACE_RESUME, **kw)
    streamed = GF.trace_symplectic(spec.mass, spec.charge, *a, chi, dt, nsteps, **kw)  # 4096 slots, one call
    GF.set_option(G.GC_OPT_WAVE_PARTICLES, 0)
    torch.cuda.synchronize()
    assert torch.equal(streamed.status, one.status) and torch.equal(streamed.n_steps, one.n_steps)
    assert torch.equal(streamed.y, one.y) and torch.equal(streamed.t, one.t)
    assert torch.equal(two.status, one.status) and torch.equal(two.n_steps, one.n_steps)
    assert rel_diff(two.y.cpu().numpy(), one.y.cpu().numpy(), spec.v_ref).max() < 1e-12   # v_par -> p_zeta -> v_par at the hand-over
    st = one.status.cpu().numpy()
    assert (st == 0).any() and ((st == 1).any() or (st == 2).any())
    idx = np.random.default_rng(11).choice(n, 96, replace=False)
    idx = np.union1d(idx, np.nonzero(st != 0)[0][:16])
    o = OF.trace_symplectic(spec.mass, spec.charge, P.s[idx], P.theta[idx], P.zeta[idx], P.vpar[idx], mu[idx], _chi(fld),
                            dt, nsteps, **kw)
    assert np.array_equal(st[idx], o.status) and np.array_equal(one.n_steps.cpu().numpy()[idx], o.n_steps)
    assert rel_diff(streamed.y.cpu().numpy()[:, idx], o.y, spec.v_ref).max() < 1e-9

