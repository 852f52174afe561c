"""Pins for the oracle's trace loop: stop rules (O7), minimum-step control (O6), end clip, Poincare
records (O8), against closed forms and properties.  CPU only."""
import math

import numpy as np

import oracle
from paper_2605_16734_b200 import workloads as W

M, Q, VREF = W.ALPHA_MASS, W.ALPHA_CHARGE, W.V_ALPHA
TWO_PI = 2.0 * math.pi


def _b00_field(ns=21, iota=0.5):
    return W.Field(ns=ns, nfp=4, xm=np.zeros(1, np.int32), xn=np.zeros(1, np.int32),
                   bmnc=np.full((ns, 1), 5.7), G=np.full(ns, 57.0), I=np.zeros(ns),
                   iota=np.full(ns, iota), psi0=W.PSI0)


def _exb_drift_field(A=-8.0e3, omega=TWO_PI * 1e3):
    """B = B00, G const, I = 0, iota = 1/2 and one mode (m, n) = (2, 1): iota m - n = 0, so alpha = 0 and
    the motion is the pure E x B drift of Phi = A sin(2 theta - zeta + omega t):
      psi(t) = psi(0) - (m A / omega) [sin(phi0 + omega t) - sin(phi0)],  v_par constant,
      zeta = zeta0 + v B t / G,  theta = theta0 + iota v B t / G   (closed form)."""
    fld = _b00_field()
    fld.mode_m = np.array([2], np.int32)
    fld.mode_n = np.array([1], np.int32)
    fld.mode_omega = np.array([omega])
    fld.mode_phase = np.array([0.0])
    fld.phihat = np.full((fld.ns, 1), A)
    return fld


def test_loss_time_against_closed_form_drift():
    A, om = -8.0e3, TWO_PI * 1e3
    fld = _exb_drift_field(A, om)
    F = oracle.OracleField(fld)
    s0 = np.array([0.9, 0.9, 0.5])
    th0 = np.array([0.1, 0.1, 0.1])
    ze0 = np.array([0.2, -0.3, 0.2])
    v0 = np.array([0.7, -0.6, 0.7]) * VREF
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / 5.7
    spec = W.make_spec(0)
    spec.t_max = 1e-4
    r = F.trace(spec, s0, th0, ze0, v0, mu, traj_capacity=5000)
    phi0 = 2 * th0 - ze0
    psi = lambda t: fld.psi0 * s0 - (2 * A / om) * (np.sin(phi0 + om * t) - np.sin(phi0))
    # particles 0 and 1 drift outward and are lost; particle 2 starts deep inside and survives
    assert list(r.status) == [1, 1, 0]
    assert r.t[2] == spec.t_max
    for i in (0, 1):
        t_star = (math.asin(math.sin(phi0[i]) - om * fld.psi0 * (1.0 - s0[i]) / (2 * A)) - phi0[i]) / om
        tr = r.traj[i, :r.traj_count[i]]
        assert tr[-1, 0] == r.t[i] and tr[-1, 1] >= 1.0          # stops on the first accepted step beyond
        assert len(tr) < 2 or tr[-2, 1] < 1.0
        assert r.t[i] >= t_star * (1 - 1e-9)
        assert len(tr) < 2 or tr[-2, 0] <= t_star * (1 + 1e-9)   # loss time = end of the crossing step (A8)
    s_exact = psi(r.t) / fld.psi0
    assert np.allclose(r.y[0], s_exact, rtol=2e-9, atol=0)
    assert np.allclose(r.y[3], v0, rtol=1e-12)
    assert np.allclose(r.y[2], ze0 + v0 * 5.7 * r.t / 57.0, rtol=1e-9)
    assert np.allclose(r.y[1], th0 + 0.5 * v0 * 5.7 * r.t / 57.0, rtol=1e-9)


def test_axis_stop_and_stop_order():
    A, om = 8.0e3, TWO_PI * 1e3                                   # inward drift for the same phases
    fld = _exb_drift_field(A, om)
    F = oracle.OracleField(fld)
    spec = W.make_spec(0)
    spec.t_max, spec.s_min = 1e-4, 0.05
    v0 = np.array([0.7 * VREF])
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / 5.7
    r = F.trace(spec, [0.1], [0.1], [0.2], v0, mu)
    assert r.status[0] == 2 and r.y[0, 0] <= 0.05 and r.t[0] < spec.t_max
    # a particle that starts beyond s_loss is reported lost after its first accepted step
    r = F.trace(spec, [1.2], [0.1], [0.2], v0, mu)
    assert r.status[0] == 1 and r.n_acc[0] == 1


def test_axis_stop_at_closed_form_time_and_start_at_or_below_s_min():
    """O7 / A7: a particle stops with status 2 on the first accepted step that ends at s <= s_min (the radial
    coordinate is singular on the axis), checked after the loss test and before the t_max test.  Inward E x B drift
    in closed form: psi(t) = psi0 s0 - (2 A / omega) (sin(phi0 + omega t) - sin(phi0)) reaches psi0 s_min at t*; the
    stopping step must straddle t*, i.e. the step before it ends above s_min (a stop rule that waits for s < 0, or
    any later s, would take further steps below s_min first)."""
    A, om = 8.0e3, TWO_PI * 1e3
    fld = _exb_drift_field(A, om)
    F = oracle.OracleField(fld)
    spec = W.make_spec(0)
    spec.t_max, spec.s_min = 1e-4, 0.05
    v0 = np.array([0.7, -0.6]) * VREF
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / 5.7
    s0, th0, ze0 = np.array([0.1, 0.12]), np.array([0.1, 0.1]), np.array([0.2, -0.3])
    r = F.trace(spec, s0, th0, ze0, v0, mu, traj_capacity=5000)
    phi0 = 2 * th0 - ze0
    assert list(r.status) == [2, 2]
    for i in range(2):
        t_star = (math.asin(math.sin(phi0[i]) + om * fld.psi0 * (s0[i] - spec.s_min) / (2 * A)) - phi0[i]) / om
        assert 0.0 < t_star < spec.t_max
        tr = r.traj[i, :r.traj_count[i]]
        assert len(tr) >= 3 and tr[-1, 0] == r.t[i] and tr[-1, 1] == r.y[0, i] <= spec.s_min
        assert tr[-2, 1] > spec.s_min                              # the step before the stop ended above s_min
        assert tr[-2, 0] <= t_star * (1 + 1e-9) and r.t[i] >= t_star * (1 - 1e-9)
        s_exact = s0[i] - (2 * A / om) * (math.sin(phi0[i] + om * r.t[i]) - math.sin(phi0[i])) / fld.psi0
        assert abs(r.y[0, i] - s_exact) < 1e-9 and r.y[0, i] > 0.0   # stopped at s_min, well before s = 0
    # a start at or below s_min stops after its first accepted step (here s stays positive: only s <= s_min says stop);
    # a start just above it does not; a start at s_loss is lost, and loss is tested before the axis
    spec.s_min = 1e-3
    fld0 = _b00_field()
    F0 = oracle.OracleField(fld0)
    v1 = np.full(4, 0.7 * VREF)
    mu1 = 0.5 * M * (VREF ** 2 - v1 ** 2) / 5.7
    r = F0.trace(spec, [5e-4, 1e-3, 2e-3, 1.0], [0.1] * 4, [0.2] * 4, v1, mu1, t_max=2e-6)
    assert list(r.status) == [2, 2, 0, 1] and list(r.n_acc[[0, 1, 3]]) == [1, 1, 1] and r.n_acc[2] > 1
    assert np.all(r.y[0, :2] > 0.0) and r.t[2] == 2e-6 and np.all(r.t[[0, 1, 3]] < 2e-6)


def test_t_max_landing_max_steps_and_start_beyond_t_max():
    F = oracle.OracleField(W.make_field(0))
    P = W.make_particles(0).head(16)
    B = F.eval_B_many(P.s, P.theta, P.zeta)[:, 0]
    mu = W.mu_from(P, B)
    spec = W.make_spec(0)
    spec.t_max = 3.3e-6
    r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    assert np.all(r.status == 0) and np.all(r.t == spec.t_max)     # exact landing (end clip)
    assert np.all(r.h > 0)
    spec.max_steps = 7
    r2 = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    assert np.all(r2.status == 3) and np.all(r2.n_acc + r2.n_rej == 7) and np.all(r2.t < spec.t_max)
    spec.max_steps = 10 ** 9
    r3 = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t0=5e-6, t_max=5e-6)
    assert np.all(r3.status == 0) and np.all(r3.n_acc == 0) and np.allclose(r3.y[0], P.s)


def test_minimum_step_control_forces_acceptance():
    """A9: with h_min far above the natural step every rejection is followed by a forced accept at h_min."""
    F = oracle.OracleField(W.make_field(0))
    P = W.make_particles(0).head(6)
    B = F.eval_B_many(P.s, P.theta, P.zeta)[:, 0]
    mu = W.mu_from(P, B)
    spec = W.make_spec(0)
    spec.t_max, spec.h_min, spec.h0 = 2e-5, 4e-7, 1e-9            # natural step is ~3e-8
    r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, traj_capacity=200)
    assert np.all(r.n_forced > 0)
    assert np.all(r.n_rej <= r.n_forced + 1)
    for i in range(P.n):
        tr = r.traj[i, :r.traj_count[i]]
        dt = np.diff(np.concatenate([[0.0], tr[:, 0]]))
        assert np.all(dt[:-1] >= spec.h_min * (1 - 1e-12))         # no step below h_min (last one is clipped)
    assert np.all(r.n_acc <= math.ceil(spec.t_max / spec.h_min) + 1)
    # h_min = 0 disables the rule
    spec.h_min = 0.0
    r0 = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    assert np.all(r0.n_forced == 0) and np.all(r0.n_acc > 100)


def test_segmented_trace_agrees_with_single_call():
    F = oracle.OracleField(W.make_field(0))
    P = W.make_particles(0).head(8)
    B = F.eval_B_many(P.s, P.theta, P.zeta)[:, 0]
    mu = W.mu_from(P, B)
    spec = W.make_spec(0)
    spec.t_max = 2e-5
    spec.rtol = spec.atol = 1e-11
    full = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    a = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=1e-5)
    b = F.trace(spec, a.y[0], a.y[1], a.y[2], a.y[3], mu, h_in=a.h, t0=1e-5, t_max=2e-5)
    scale = np.array([[1.0], [1.0], [1.0], [VREF]])
    assert (np.abs(b.y - full.y) / scale).max() < 1e-8
    assert np.all(a.h > 5e-9)          # the clipped last step did not poison the carried step size


def test_poincare_crossings_closed_form_both_directions():
    """O8 on case (c): zeta = zeta0 + v B00 t / G, so the planes zeta = 2 pi k are crossed at
    t_k = (2 pi k - zeta0) G / (v B00) with theta_k = theta0 + iota (2 pi k - zeta0), s unchanged."""
    fld = _b00_field(iota=0.47)
    F = oracle.OracleField(fld)
    s0 = np.array([0.3, 0.6]); th0 = np.array([0.5, 1.0]); ze0 = np.array([0.1, -2.0])
    v0 = np.array([0.8, -0.5]) * VREF
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / 5.7
    spec = W.make_spec(0)
    spec.t_max = 4e-5
    r = F.trace(spec, s0, th0, ze0, v0, mu, poincare_capacity=1000)
    rate = v0 * 5.7 / 57.0
    expected = []
    for i in range(2):
        ze_end = ze0[i] + rate[i] * spec.t_max
        ks = (range(1, math.floor(ze_end / TWO_PI) + 1) if rate[i] > 0
              else range(math.floor(ze0[i] / TWO_PI), math.floor(ze_end / TWO_PI), -1))
        for k in ks:
            tk = (TWO_PI * k - ze0[i]) / rate[i]
            expected.append((i, tk, s0[i], (th0[i] + 0.47 * (TWO_PI * k - ze0[i])) % TWO_PI))
    assert r.poincare_count == len(expected) and len(expected) >= 8
    got = r.poincare[np.lexsort((r.poincare[:, 1], r.poincare[:, 0]))]
    exp = np.array(sorted(expected))
    assert np.array_equal(got[:, 0], exp[:, 0])
    assert np.allclose(got[:, 1], exp[:, 1], rtol=1e-10)
    assert np.allclose(got[:, 2], exp[:, 2], rtol=1e-12)
    dth = np.abs(got[:, 3] - exp[:, 3])
    assert np.all(np.minimum(dth, TWO_PI - dth) < 1e-9)
    # overflow is signalled by count > capacity, excess dropped
    r2 = F.trace(spec, s0, th0, ze0, v0, mu, poincare_capacity=5)
    assert r2.poincare_count == len(expected) and len(r2.poincare) == 5


def test_config0_workload_shape():
    """The synthetic ensemble behaves like the paper's workloads: step sizes, rejection ratio, prompt losses
    (SURVEY.md section 8(d) 'workload structure')."""
    F = oracle.OracleField(W.make_field(0))
    P = W.make_particles(0).head(48)
    B = F.eval_B_many(P.s, P.theta, P.zeta)[:, 0]
    mu = W.mu_from(P, B)
    spec = W.make_spec(0)
    r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    assert set(np.unique(r.status)) <= {0, 1}
    rej = r.n_rej.sum() / (r.n_acc.sum() + r.n_rej.sum())
    assert 0.03 < rej < 0.4
    per_s = r.n_acc.sum() / r.t.sum()
    assert 5e6 < per_s < 2e8


def test_refined_loss_time_against_closed_form_drift():
    """O7b: with refine_loss the loss time is the root of s(tau) = s_loss on the continuous extension, which in the
    E x B drift field has a closed form; the reported state sits on the boundary; survivors and the rest of the
    trace are untouched."""
    A, om = -8.0e3, TWO_PI * 1e3
    fld = _exb_drift_field(A, om)
    F = oracle.OracleField(fld)
    s0 = np.array([0.9, 0.9, 0.5])
    th0 = np.array([0.1, 0.1, 0.1])
    ze0 = np.array([0.2, -0.3, 0.2])
    v0 = np.array([0.7, -0.6, 0.7]) * VREF
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / 5.7
    spec = W.make_spec(0)
    spec.t_max = 1e-4
    a = F.trace(spec, s0, th0, ze0, v0, mu)
    r = F.trace(spec, s0, th0, ze0, v0, mu, refine_loss=True)
    phi0 = 2 * th0 - ze0
    assert list(r.status) == [1, 1, 0]
    assert np.array_equal(r.n_acc, a.n_acc) and np.array_equal(r.n_rej, a.n_rej)
    assert np.array_equal(r.y[:, 2], a.y[:, 2]) and r.t[2] == a.t[2]
    for i in (0, 1):
        t_star = (math.asin(math.sin(phi0[i]) - om * fld.psi0 * (1.0 - s0[i]) / (2 * A)) - phi0[i]) / om
        assert abs(r.t[i] - t_star) < 2e-7 * t_star              # accuracy of the 4th-order extension, not the step size
        assert abs(a.t[i] - t_star) > 1e-6 * t_star              # the unrefined time is a step end
        assert r.t[i] <= a.t[i] and abs(r.y[0, i] - 1.0) < 1e-13
        assert np.isclose(r.y[2, i], ze0[i] + v0[i] * 5.7 * r.t[i] / 57.0, rtol=1e-9)
        assert np.isclose(r.y[3, i], v0[i], rtol=1e-12)
