"""Pins of the oracle's NEXT-1 pieces: O9 uniform-time samples of the
Dormand-Prince continuous extension ("dense output"), P_zeta along them (A17), and the
weighted Birkhoff average with its digit accuracy.  Nothing here comes from the CUDA path."""
from __future__ import annotations

import math

import numpy as np
import pytest
from scipy.integrate import solve_ivp

import oracle
from paper_2605_16734_b200 import workloads as W

M, Q, VREF = W.ALPHA_MASS, W.ALPHA_CHARGE, W.V_ALPHA


def _mu_for(F, P):
    B = F.eval_B_many(P.s, P.theta, P.zeta)[:, 0]
    return W.mu_from(P, B)


# ---- O9: samples -----------------------------------------------------------------------------------------------
def test_samples_of_closed_form_passing_orbit():
    """Only B00 and constant iota, I = 0: s and v_par stay, zeta = zeta0 + v B00 t / G, theta = theta0 + iota v B00
    t / G.  Runge-Kutta and its continuous extension are exact on linear motion, so every sample is the closed
    form to rounding; all nsamp samples are written, the first one (tau_0 = t0) is the initial state."""
    ns = 21
    s_n = np.arange(ns) / (ns - 1)
    fld = W.Field(ns=ns, nfp=4, xm=np.zeros(1, np.int32), xn=np.zeros(1, np.int32), bmnc=np.full((ns, 1), 5.7),
                  G=np.full(ns, 57.0), I=np.zeros(ns), iota=0.42 + 0.1 * s_n, psi0=W.PSI0)
    F = oracle.OracleField(fld)
    s0 = np.array([0.3, 0.6]); th0 = np.array([0.5, 1.0]); ze0 = np.array([0.1, -2.0])
    v0 = np.array([0.8, -0.5]) * VREF
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / 5.7
    spec = W.make_spec(0)
    spec.t_max = 2e-5
    nsamp, dt = 41, 5e-7                                   # tau_40 = 2e-5 = t_max: the last sample is the end state
    r = F.trace_sampled(spec, s0, th0, ze0, v0, mu, 0.0, dt, nsamp)
    assert np.all(r.nsampled == nsamp)
    tau = dt * np.arange(nsamp)
    io = 0.42 + 0.1 * s0
    for i in range(2):
        assert np.allclose(r.samples[0, :, i], s0[i], rtol=1e-13)
        assert np.allclose(r.samples[3, :, i], v0[i], rtol=1e-13)
        assert np.allclose(r.samples[2, :, i], ze0[i] + v0[i] * 5.7 * tau / 57.0, rtol=1e-12, atol=1e-13)
        assert np.allclose(r.samples[1, :, i], th0[i] + io[i] * v0[i] * 5.7 * tau / 57.0, rtol=1e-12, atol=1e-13)
    assert np.array_equal(r.samples[:, 0, :], np.stack([s0, th0, ze0, v0]))
    # the sampled trace is the plain trace: same end state, same step counts
    r0 = F.trace(spec, s0, th0, ze0, v0, mu)
    assert np.array_equal(r0.y, r.y) and np.array_equal(r0.n_acc, r.n_acc) and np.array_equal(r0.n_rej, r.n_rej)


def test_samples_match_an_independent_integration():
    """Config 0: the samples agree with scipy's DOP853 (rtol 1e-12) of the oracle's right-hand side at the same
    times to the accuracy of the 4th-order continuous extension at rtol 1e-9; the error shrinks with rtol."""
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    P = W.make_particles(0).head(4)
    mu = _mu_for(F, P)
    nsamp, dt = 33, 6.25e-8
    tau = dt * np.arange(nsamp)
    errs = {}
    for rtol in (1e-7, 1e-9):
        spec = W.make_spec(0)
        spec.rtol = spec.atol = rtol
        spec.t_max = 2e-6
        r = F.trace_sampled(spec, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, dt, nsamp)
        assert np.all(r.nsampled == nsamp)
        worst = 0.0
        for i in range(P.n):
            f = lambda t, y: F.rhs(M, Q, mu[i], VREF, t, y)
            sol = solve_ivp(f, (0.0, spec.t_max), [P.s[i], P.theta[i], P.zeta[i], P.vpar[i] / VREF],
                            method="DOP853", rtol=1e-12, atol=1e-14, t_eval=tau)
            ref = sol.y.copy()
            ref[3] *= VREF
            got = r.samples[:, :, i]
            scale = np.array([1.0, 1.0, 1.0, VREF])[:, None]
            worst = max(worst, float(np.abs((got - ref) / scale).max()))
        errs[rtol] = worst
    assert errs[1e-9] < 1e-7                               # the extension is one order below the step itself
    assert errs[1e-9] < 0.1 * errs[1e-7]


def test_samples_stop_with_the_particle_and_sample_grid_may_start_anywhere():
    """A lost particle leaves the samples after its loss time untouched (NaN fill of the wrapper); a sample grid that
    starts before t0 or between steps is entered at the first tau_j >= t0."""
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    P = W.make_particles(0).head(8)
    mu = _mu_for(F, P)
    spec = W.make_spec(0)
    spec.s_loss = 0.2502                                   # particles start on s = 0.25: some are "lost" at once
    spec.t_max = 4e-6
    nsamp, dt = 40, 1e-7
    r = F.trace_sampled(spec, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, dt, nsamp)
    assert (r.status == 1).any() and (r.status == 0).any()
    for i in range(P.n):
        k = int(r.nsampled[i])
        assert k == min(nsamp, int(math.floor(r.t[i] / dt + 1e-9)) + 1)      # tau_0 .. tau_{k-1} <= t_out
        assert np.isfinite(r.samples[:, :k, i]).all() and np.isnan(r.samples[:, k:, i]).all()
    # grid shifted by -2.5 dt: tau_j = (j - 2.5) dt; the first sample at or after t0 = 0 is j = 3
    spec.s_loss = 1.0
    r2 = F.trace_sampled(spec, P.s, P.theta, P.zeta, P.vpar, mu, -2.5 * dt, dt, nsamp)
    assert np.isnan(r2.samples[:, :3, :]).all() and np.isfinite(r2.samples[:, 3:, :]).all()
    assert np.all(r2.nsampled == nsamp)


def test_samples_over_two_segments():
    """Segments (t0 -> t1 -> t2, carrying h) on a grid whose points are exact in binary: the first call writes
    tau_0 .. tau_8 = t1, the second re-writes tau_8 (a sample on its t0 is its initial state: the same values) and
    continues with tau_9 .. tau_16; nothing else is touched; the two-segment series agrees with one call over
    [t0, t2] to the integrator's accuracy (the end clip at t1 changes the step sequence)."""
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    P = W.make_particles(0).head(5)
    mu = _mu_for(F, P)
    spec = W.make_spec(0)
    dt, nsamp = 2.0 ** -23, 17
    t1, t2 = 8 * dt, 16 * dt
    a = F.trace_sampled(spec, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, dt, nsamp, t0=0.0, t_max=t1)
    assert np.all(a.nsampled == 9)
    assert np.isfinite(a.samples[:, :9, :]).all() and np.isnan(a.samples[:, 9:, :]).all()
    assert np.array_equal(a.samples[:, 8, :], a.y)        # tau_8 = t_max exactly: tau = 1 of the last step
    b = F.trace_sampled(spec, a.y[0], a.y[1], a.y[2], a.y[3], mu, 0.0, dt, nsamp, h_in=a.h, t0=t1, t_max=t2)
    assert np.all(b.nsampled == 17)
    assert np.isnan(b.samples[:, :8, :]).all() and np.isfinite(b.samples[:, 8:, :]).all()
    assert np.array_equal(b.samples[:, 8, :], a.y)
    one = F.trace_sampled(spec, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, dt, nsamp, t0=0.0, t_max=t2)
    both = np.where(np.isnan(b.samples), a.samples, b.samples)
    scale = np.array([1.0, 1.0, 1.0, VREF])[:, None, None]
    assert np.abs((both - one.samples) / scale).max() < 1e-7


# ---- A17: P_zeta along the samples ---------------------------------------------------------------------------------
def test_pzeta_of_samples_is_conserved_in_an_axisymmetric_field():
    """remove the non-symmetric harmonics and the canonical momentum is conserved.  Evaluated with
    oracle_pzeta on the uniform-time samples (iota linear in s, so chi at the nodes is exact and its cubic
    interpolation too); it really is P_zeta that is constant: s moves by > 0.01."""
    fld = W.make_field(0)
    keep = fld.xn == 0
    fld.xm, fld.xn, fld.bmnc = fld.xm[keep], fld.xn[keep], np.ascontiguousarray(fld.bmnc[:, keep])
    F = oracle.OracleField(fld)
    s_n = np.arange(fld.ns) / (fld.ns - 1)
    chi_nodes = fld.psi0 * (0.42 * s_n + 0.05 * s_n ** 2)
    P = W.make_particles(0).head(6)
    mu = _mu_for(F, P)
    spec = W.make_spec(0)
    nsamp, dt = 101, 1e-6                                  # 1e-4 s, the protocol of the paper's Fig. 1 right
    r = F.trace_sampled(spec, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, dt, nsamp)
    assert np.all(r.nsampled == nsamp)
    tau = dt * np.arange(nsamp)
    moved = 0.0
    for i in range(P.n):
        sm = r.samples[:, :, i]
        pz = F.pzeta(M, Q, chi_nodes, sm[0], sm[1], sm[2], sm[3], tau)
        assert np.abs(pz / pz[0] - 1.0).max() < 1e-7
        moved = max(moved, np.ptp(sm[0]))
    assert moved > 0.01
    # a wrong sign or a missing term shows at once: P_zeta without the chi term is NOT constant
    pz_bad = F.pzeta(M, Q, np.zeros(fld.ns), sm[0], sm[1], sm[2], sm[3], tau)
    assert np.abs(pz_bad / pz_bad[0] - 1.0).max() > 1e-4


def test_pzeta_with_modes_n_H_minus_omega_P_zeta():
    """Axisymmetric equilibrium + modes sharing n and omega: n H - omega P_zeta is exact while P_zeta itself varies;
    pins the alpha term of oracle_pzeta (H is assembled here from the oracle's B and Phi)."""
    fld = W.make_field(0)
    s_n = np.arange(fld.ns) / (fld.ns - 1)
    amp = fld.bmnc[-1, :].copy()
    fld.bmnc = np.ascontiguousarray(amp[None, :] * (0.2 * s_n + 0.8 * s_n ** 2 - 0.3 * s_n ** 3)[:, None])
    fld.bmnc[:, 0] = 5.7
    keep = fld.xn == 0
    fld.xm, fld.xn, fld.bmnc = fld.xm[keep], fld.xn[keep], np.ascontiguousarray(fld.bmnc[:, keep])
    fld.mode_m = np.array([3, 4], np.int32)
    fld.mode_n = np.array([2, 2], np.int32)
    fld.mode_omega = np.full(2, 2 * math.pi * 120e3)
    fld.mode_phase = np.array([0.0, 1.0])
    env = 4.0 * (s_n - s_n ** 3)
    fld.phihat = np.stack([4e4 * env, -3e4 * env], axis=1)
    F = oracle.OracleField(fld)
    chi_nodes = fld.psi0 * (0.42 * s_n + 0.05 * s_n ** 2)
    P = W.make_particles(0).head(4)
    mu = _mu_for(F, P)
    spec = W.make_spec(0)
    spec.rtol = spec.atol = 1e-11
    spec.t_max = 5e-5
    nsamp, dt = 51, 1e-6
    r = F.trace_sampled(spec, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, dt, nsamp)
    tau = dt * np.arange(nsamp)
    varied = 0.0
    for i in range(P.n):
        sm = r.samples[:, :, i]
        pz = F.pzeta(M, Q, chi_nodes, sm[0], sm[1], sm[2], sm[3], tau)
        H = np.array([0.5 * M * sm[3, j] ** 2 + mu[i] * F.eval_B(sm[0, j], sm[1, j], sm[2, j])[0]
                      + Q * F.eval_pert(sm[0, j], sm[1, j], sm[2, j], tau[j])[0] for j in range(nsamp)])
        inv = 2.0 * H - fld.mode_omega[0] * pz
        ref = abs(2.0 * H[0]) + abs(fld.mode_omega[0] * pz[0])
        assert np.abs(inv - inv[0]).max() < 1e-8 * ref       # samples carry the 4th-order extension's error
        varied = max(varied, np.abs(pz / pz[0] - 1.0).max())
    assert varied > 1e-6


# ---- weighted Birkhoff average --------------------------------------------------------------------------------------
def test_birkhoff_weights_and_average_basics():
    w = oracle.birkhoff_weights(1001)
    assert np.all(w >= 0.0) and np.all(w[1:-1] > 0.0) and np.allclose(w, w[::-1], rtol=1e-12)   # symmetric bump
    assert w[500] == pytest.approx(math.exp(-4.0), rel=1e-12)               # g(1/2) = exp(-1/(1/4))
    assert w[0] < 1e-300 and np.all(np.diff(w[:501]) >= 0.0)                # flat to all orders at the ends
    rng = np.random.default_rng(7)
    f, g = rng.standard_normal(400), rng.standard_normal(400)
    assert oracle.birkhoff_average(np.full(400, 2.5)) == pytest.approx(2.5, rel=1e-15)
    assert oracle.birkhoff_average(3.0 * f - 2.0 * g) == pytest.approx(
        3.0 * oracle.birkhoff_average(f) - 2.0 * oracle.birkhoff_average(g), rel=1e-12, abs=1e-14)
    # brute force on a tiny series
    x = (np.arange(5) + 1.0) / 6.0
    ww = [math.exp(-1.0 / (xi * (1.0 - xi))) for xi in x]
    assert oracle.birkhoff_average([1.0, 2.0, 4.0, 8.0, 16.0]) == pytest.approx(
        sum(a * b for a, b in zip(ww, [1.0, 2.0, 4.0, 8.0, 16.0])) / sum(ww), rel=1e-14)


def test_birkhoff_superconvergence_on_a_quasiperiodic_signal():
    """The property the method exists for: for f(j) = c + sum_k a_k cos(2 pi k nu j + p_k) with Diophantine nu the
    weighted average converges to c faster than any power of N, the plain mean only like 1/N."""
    nu = 0.5 * (math.sqrt(5.0) - 1.0)
    j = np.arange(4000)
    f = 1.75 + 0.8 * np.cos(2 * np.pi * nu * j + 0.3) - 0.4 * np.cos(2 * np.pi * 3 * nu * j + 1.1)
    assert abs(oracle.birkhoff_average(f) - 1.75) < 1e-12
    assert abs(np.mean(f) - 1.75) > 1e-6
    e500, e2000 = abs(oracle.birkhoff_average(f[:500]) - 1.75), abs(oracle.birkhoff_average(f[:2000]) - 1.75)
    assert e500 < 1e-5 and e2000 < 1e-3 * max(e500, 1e-13) + 1e-13          # far faster than 1/N


def test_birkhoff_digits_separate_regular_from_chaotic():
    """Digit accuracy (below 3 indicates chaotic motion): a quasi-periodic series gives > 10 digits,
    the logistic map at r = 4 (chaotic, invariant mean 1/2) gives < 3."""
    nu = math.sqrt(2.0) - 1.0
    j = np.arange(6000)
    a, b, d = oracle.birkhoff_digits(2.0 + np.sin(2 * np.pi * nu * j))
    assert d > 10.0 and a == pytest.approx(2.0, abs=1e-10) and b == pytest.approx(2.0, abs=1e-10)
    x = np.empty(6000)
    x[0] = 0.123456
    for k in range(1, 6000):
        x[k] = 4.0 * x[k - 1] * (1.0 - x[k - 1])
    a, b, d = oracle.birkhoff_digits(x)
    assert d < 3.0 and abs(a - 0.5) < 0.1 and abs(b - 0.5) < 0.1
    assert oracle.birkhoff_digits(np.full(100, 3.0))[2] == 16.0
    # invariant under scaling of the signal
    assert oracle.birkhoff_digits(7.0 * x)[2] == pytest.approx(d, abs=1e-9)


# ---- O8b: bounce section v_par = 0 -----------------------------------------------------------------------------------
def test_bounce_section_matches_event_location_of_an_independent_integrator():
    """Trapped particles of config 0: every record of the v_par = 0 section agrees in time and position with the
    events scipy's DOP853 (rtol 1e-12, dense output + root finding) locates on the oracle's right-hand side; the
    number of records is the number of sign changes of v_par along the accepted steps; passing particles give none."""
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    P = W.make_particles(0).head(40)
    mu = _mu_for(F, P)
    spec = W.make_spec(0)
    spec.t_max = 4e-5
    r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, poincare_capacity=4000, traj_capacity=20000, section=1)
    rec = r.poincare[np.lexsort((r.poincare[:, 1], r.poincare[:, 0]))]
    assert r.poincare_count == len(rec) > 20
    per = {i: rec[rec[:, 0] == i] for i in range(P.n)}
    checked = 0
    for i in range(P.n):
        tr = r.traj[i, :r.traj_count[i]]
        u = np.concatenate([[P.vpar[i] / VREF], tr[:, 4]])
        changes = int(np.sum((u[:-1] < 0) & (u[1:] >= 0)) + np.sum((u[:-1] > 0) & (u[1:] <= 0)))
        assert len(per[i]) == changes
        if changes == 0:                                       # passing, or not yet turned: no record
            continue
        if checked >= 6:
            continue
        ev = lambda t, y: y[3]
        sol = solve_ivp(lambda t, y: F.rhs(M, Q, mu[i], VREF, t, y), (0.0, float(r.t[i])),
                        [P.s[i], P.theta[i], P.zeta[i], P.vpar[i] / VREF], method="DOP853", rtol=1e-12, atol=1e-14,
                        events=ev)
        te, ye = sol.t_events[0], sol.y_events[0]
        te, ye = te[te > 0], ye[te > 0]
        assert len(te) == changes
        assert np.abs(per[i][:, 1] - te).max() < 1e-11          # seconds; bounce periods are ~1e-5 s
        assert np.abs(per[i][:, 2] - ye[:, 0]).max() < 2e-6     # global error of the rtol 1e-9 trace after ~30 bounces
        dth = np.abs(per[i][:, 3] - np.mod(ye[:, 1], 2 * np.pi))
        assert np.minimum(dth, 2 * np.pi - dth).max() < 2e-5
        checked += 1
    assert checked >= 4
    passing = [i for i in range(P.n) if abs(P.vpar[i]) / VREF > 0.8]
    assert passing and all(len(per[i]) == 0 for i in passing)


def test_bounce_section_in_a_closed_form_field_has_no_crossings_and_zeta_section_is_unchanged():
    """B00-only field: v_par is constant, so the bounce section records nothing whatever the sign of v_par; the
    default section (zeta planes) of the same call is what it was (section = 0 is the old behaviour)."""
    ns = 21
    s_n = np.arange(ns) / (ns - 1)
    fld = W.Field(ns=ns, nfp=4, xm=np.zeros(1, np.int32), xn=np.zeros(1, np.int32), bmnc=np.full((ns, 1), 5.7),
                  G=np.full(ns, 57.0), I=np.zeros(ns), iota=0.42 + 0.1 * s_n, psi0=W.PSI0)
    F = oracle.OracleField(fld)
    s0 = np.array([0.3, 0.6]); th0 = np.array([0.5, 1.0]); ze0 = np.array([0.1, -2.0])
    v0 = np.array([0.8, -0.5]) * VREF
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / 5.7
    spec = W.make_spec(0)
    spec.t_max = 2e-5
    b = F.trace(spec, s0, th0, ze0, v0, mu, poincare_capacity=100, section=1)
    assert b.poincare_count == 0
    z = F.trace(spec, s0, th0, ze0, v0, mu, poincare_capacity=100, section=0)
    z0 = F.trace(spec, s0, th0, ze0, v0, mu, poincare_capacity=100)
    srt = lambda a: a[np.lexsort((a[:, 1], a[:, 0]))]           # record order depends on the thread schedule
    assert z.poincare_count == z0.poincare_count > 0 and np.array_equal(srt(z.poincare), srt(z0.poincare))
