"""Pins for the oracle's guiding-centre equations (O4) and trace (O5-O8) against what the mathematics fixes:
the Euler-Lagrange equations of the guiding-centre Lagrangian solved numerically, exact invariants, closed-form
orbits and a brute-force fixed-step RK4.  CPU only.  (SURVEY.md section 8(c) checks (a)-(e).)"""
import math

import numpy as np
import pytest

import oracle
from paper_2605_16734_b200 import workloads as W

M, Q, VREF = W.ALPHA_MASS, W.ALPHA_CHARGE, W.V_ALPHA


def _general_field(with_modes=True):
    """Non-trivial G(s), I(s), iota(s) and (optionally) strong modes so that every term of O4 matters."""
    fld = W.make_equilibrium(4, 4, 41)
    s = np.arange(fld.ns) / (fld.ns - 1)
    fld.G = 57.0 + 6.0 * s - 2.0 * s ** 2
    fld.I = 4.0 * s + 1.0 * s ** 2
    fld.iota = 0.42 + 0.3 * s
    if with_modes:
        fld.mode_m = np.array([3, 5, 2], np.int32)
        fld.mode_n = np.array([2, 2, -1], np.int32)
        fld.mode_omega = np.array([7.5e5, 7.5e5, -4.0e5])
        fld.mode_phase = np.array([0.0, 0.7, 2.0])
        env = np.exp(-((s - 0.45) ** 2) / (2 * 0.2 ** 2))
        fld.phihat = np.stack([3e5 * env, -2e5 * env * (1 + s), 1e5 * env ** 2], axis=1)
    return fld


def _lagrangian_rhs(F, fld, mu, t, z):
    """Solve  sum_j omega_ij zdot_j = dH/dz_i + dLambda_i/dt,  omega_ij = dLambda_j/dz_i - dLambda_i/dz_j,
    for L = Lambda_theta thdot + Lambda_zeta zedot - H with
      Lambda_theta = q (psi + rho_c I),  Lambda_zeta = q (rho_c G - chi),  chi' = iota,
      rho_c = m v/(q B) + alpha,  H = m v^2/2 + mu B + q Phi,
    all derivatives by Richardson-extrapolated central differences of the oracle's *point evaluations*."""
    psi0 = fld.psi0

    def parts(zz, tt):
        s, th, ze, v = zz
        B = F.eval_B(s, th, ze)[0]
        G, _, I, _, _, _ = F.eval_profiles(s)
        pt = F.eval_pert(s, th, ze, tt)
        rho_c = M * v / (Q * B) + pt[4]
        Lth = Q * (psi0 * s + rho_c * I)
        Lze_nochi = Q * rho_c * G                     # chi handled analytically: d chi/ds = psi0 iota
        H = 0.5 * M * v * v + mu * B + Q * pt[0]
        return np.array([Lth, Lze_nochi, H])

    steps = np.array([2e-4, 1e-3, 1e-3, 2e-3 * VREF])

    def dz(i):
        def cd(h):
            e = np.zeros(4)
            e[i] = h
            return (parts(z + e, t) - parts(z - e, t)) / (2 * h)
        h = steps[i]
        return (4.0 * cd(h / 2) - cd(h)) / 3.0          # O(h^4)

    def dt_():
        h = 2e-8
        cd = lambda hh: (parts(z, t + hh) - parts(z, t - hh)) / (2 * hh)
        return (4.0 * cd(h / 2) - cd(h)) / 3.0

    D = np.array([dz(i) for i in range(4)])             # D[i] = d(parts)/dz_i
    Dt = dt_()
    iota = F.eval_profiles(z[0])[4]
    dLth = D[:, 0].copy()
    dLze = D[:, 1].copy()
    dLze[0] -= Q * psi0 * iota
    dH = D[:, 2]
    Lam = np.zeros((4, 4))                              # Lam[j][i] = dLambda_j/dz_i ; z = (s, th, ze, v)
    Lam[1, :] = dLth
    Lam[2, :] = dLze
    omega = Lam.T - Lam                                 # omega_ij = dLambda_j/dz_i - dLambda_i/dz_j
    rhs = dH + np.array([0.0, Dt[0], Dt[1], 0.0])
    scale = np.abs(omega).max(axis=1, keepdims=True)
    return np.linalg.solve(omega / scale, rhs / scale[:, 0])


@pytest.mark.parametrize("with_modes", [False, True])
def test_rhs_equals_euler_lagrange_equations(with_modes):
    fld = _general_field(with_modes)
    F = oracle.OracleField(fld)
    rng = np.random.default_rng(7)
    for _ in range(6):
        s = (math.floor(rng.uniform(0.15, 0.85) * (fld.ns - 1)) + 0.5) / (fld.ns - 1)
        th, ze = rng.uniform(-3, 3, 2)
        v = rng.uniform(-1, 1) * VREF
        if abs(v) < 0.1 * VREF:
            v = 0.3 * VREF
        B = F.eval_B(s, th, ze)[0]
        mu = 0.5 * M * (VREF ** 2 - v ** 2) / B
        t = float(rng.uniform(0, 1e-5))
        got = F.rhs(M, Q, mu, VREF, t, [s, th, ze, v / VREF])
        got = np.array([got[0], got[1], got[2], got[3] * VREF])
        ref = _lagrangian_rhs(F, fld, mu, t, np.array([s, th, ze, v]))
        # each component against its own scale: a dropped or mis-signed term shows up at >= 1e-3
        tol = 2e-6 * np.maximum(np.abs(ref), np.array([1e-2 * abs(ref[1]), 0, 0, 1e-3 * abs(ref[3]) + 1.0]))
        assert np.all(np.abs(got - ref) <= tol + 1e-7 * np.abs(ref)), (got, ref)
    if with_modes:        # the perturbation must matter in this test, else it pins nothing
        F0 = oracle.OracleField(_general_field(False))
        base = F0.rhs(M, Q, mu, VREF, t, [s, th, ze, v / VREF])
        assert abs(got[0] - base[0]) > 1e-3 * abs(base[0])


def _mu_for(F, P):
    B = F.eval_B_many(P.s, P.theta, P.zeta)[:, 0]
    return W.mu_from(P, B), B


def _traj_arrays(res, i):
    c = int(res.traj_count[i])
    assert c <= res.traj.shape[1], "trajectory buffer too small for this test"
    return res.traj[i, :c, :]


def test_energy_and_mu_conserved_in_static_field():
    """(a) PAPER.md:62: time-independent field conserves E = m v^2/2 + mu B; RK drift bounded by tolerance."""
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    P = W.make_particles(0).head(12)
    mu, B0 = _mu_for(F, P)
    E0 = 0.5 * M * P.vpar ** 2 + mu * B0
    drift = {}
    for rtol in (1e-7, 1e-9, 1e-11):
        spec = W.make_spec(0)
        spec.rtol = spec.atol = rtol
        r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, traj_capacity=20000)
        worst = 0.0
        for i in range(P.n):
            tr = _traj_arrays(r, i)
            idx = np.linspace(0, len(tr) - 1, 40).astype(int)
            Bt = F.eval_B_many(tr[idx, 1], tr[idx, 2], tr[idx, 3])[:, 0]
            E = 0.5 * M * (tr[idx, 4] * VREF) ** 2 + mu[i] * Bt
            worst = max(worst, np.abs(E / E0[i] - 1).max())
        drift[rtol] = worst
        steps = (r.n_acc + r.n_rej).max()
        assert worst < steps * rtol
    assert drift[1e-9] < 0.05 * drift[1e-7]
    assert drift[1e-11] < 0.05 * drift[1e-9]


def _p_zeta(F, fld, tr, mu, chi):
    out = np.empty(len(tr))
    for j, (t, s, th, ze, u) in enumerate(tr):
        B = F.eval_B(s, th, ze)[0]
        G, _, I, _, _, _ = F.eval_profiles(s)
        al = F.eval_pert(s, th, ze, t)[4]
        out[j] = Q * ((M * u * VREF / (Q * B) + al) * G - chi(s))
    return out


def _p_theta(F, fld, tr):
    out = np.empty(len(tr))
    for j, (t, s, th, ze, u) in enumerate(tr):
        B = F.eval_B(s, th, ze)[0]
        G, _, I, _, _, _ = F.eval_profiles(s)
        al = F.eval_pert(s, th, ze, t)[4]
        out[j] = Q * (fld.psi0 * s + (M * u * VREF / (Q * B) + al) * I)
    return out


def test_p_zeta_conserved_in_axisymmetric_field():
    """(b) PAPER.md:60,62: symmetric field => canonical momentum conserved; protocol of Fig. 1 right
    (10 particles, 1e-4 s, max over trajectory and particles); error falls with the tolerance."""
    fld = W.make_field(0)
    keep = fld.xn == 0                                  # remove the non-symmetric harmonics
    fld.xm, fld.xn, fld.bmnc = fld.xm[keep], fld.xn[keep], np.ascontiguousarray(fld.bmnc[:, keep])
    F = oracle.OracleField(fld)
    chi = lambda s: fld.psi0 * (0.42 * s + 0.05 * s * s)
    P = W.make_particles(0).head(10)
    mu, _ = _mu_for(F, P)
    worst = {}
    for rtol in (1e-7, 1e-9, 1e-11):
        spec = W.make_spec(0)
        spec.rtol = spec.atol = rtol
        r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, traj_capacity=30000)
        w = 0.0
        moved = 0.0
        for i in range(P.n):
            tr = _traj_arrays(r, i)
            tr = tr[np.linspace(0, len(tr) - 1, 60).astype(int)]
            pz = _p_zeta(F, fld, tr, mu[i], chi)
            w = max(w, np.abs(pz / pz[0] - 1).max())
            moved = max(moved, np.ptp(tr[:, 1]))
        worst[rtol] = w
        assert moved > 0.01                             # orbits really move radially
    assert worst[1e-9] < 1e-7                           # paper quotes ~1e-8 at tol 1e-9 (context)
    # falls with the tolerance until the kinks of the piecewise-cubic interpolant at the radial nodes set
    # a floor (the paper's Fig. 1 right shows the same dependence on the node count)
    assert worst[1e-9] < 0.1 * worst[1e-7]
    assert worst[1e-11] < 0.3 * worst[1e-9]


def test_helical_momentum_conserved_in_quasihelical_field():
    """(b') harmonics (m, n) = j (1, 1): B depends on theta - nfp*zeta only, so
    P_zeta + nfp * P_theta is conserved (A17), with I != 0 so that P_theta's rho term is exercised."""
    fld = W.make_field(0)
    keep = (fld.xm == fld.xn)
    fld.xm, fld.xn, fld.bmnc = fld.xm[keep], fld.xn[keep], np.ascontiguousarray(fld.bmnc[:, keep])
    assert keep.sum() == 9
    s = np.arange(fld.ns) / (fld.ns - 1)
    fld.I = 3.0 * s
    F = oracle.OracleField(fld)
    chi = lambda s_: fld.psi0 * (0.42 * s_ + 0.05 * s_ * s_)
    P = W.make_particles(0).head(6)
    mu, _ = _mu_for(F, P)
    spec = W.make_spec(0)
    spec.rtol = spec.atol = 1e-11
    r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, traj_capacity=40000)
    for i in range(P.n):
        tr = _traj_arrays(r, i)
        tr = tr[np.linspace(0, len(tr) - 1, 50).astype(int)]
        pz, pth = _p_zeta(F, fld, tr, mu[i], chi), _p_theta(F, fld, tr)
        inv = pz + fld.nfp * pth
        assert np.abs(inv / inv[0] - 1).max() < 1e-9
        assert np.abs(pz / pz[0] - 1).max() > 1e-4      # while P_zeta alone is not conserved


def test_closed_form_passing_orbit():
    """(c) only B00(s) = b0 + b1 s, linear G, I, iota: sdot = vdot = 0 and constant angular rates (O4).
    With b1 = 0, I = 0: zeta = zeta0 + v B00 t / G, theta = theta0 + iota v B00 t / G."""
    ns = 21
    s_n = np.arange(ns) / (ns - 1)
    for b1, I1 in ((0.0, 0.0), (0.6, 2.0)):
        fld = W.Field(ns=ns, nfp=4, xm=np.zeros(1, np.int32), xn=np.zeros(1, np.int32),
                      bmnc=(5.7 + b1 * s_n)[:, None].copy(), G=57.0 + 1.5 * s_n * (b1 != 0), I=I1 * s_n,
                      iota=0.42 + 0.1 * s_n, psi0=W.PSI0)
        F = oracle.OracleField(fld)
        s0 = np.array([0.3, 0.6]); th0 = np.array([0.5, 1.0]); ze0 = np.array([0.1, -2.0])
        v0 = np.array([0.8, -0.5]) * VREF
        B = 5.7 + b1 * s0
        mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / B
        spec = W.make_spec(0)
        spec.t_max = 2e-5
        r = F.trace(spec, s0, th0, ze0, v0, mu)
        assert np.all(r.status == 0) and np.all(r.t == spec.t_max)
        # rates from O4 with constant coefficients
        G = 57.0 + 1.5 * s0 * (b1 != 0); Gp = (1.5 * (b1 != 0)) / fld.psi0
        I = I1 * s0; Ip = I1 / fld.psi0; io = 0.42 + 0.1 * s0
        rho = M * v0 / (Q * B); Fm = M * v0 ** 2 / B + mu; Bp = b1 / fld.psi0
        D = G + io * I + rho * (G * Ip - I * Gp)
        thd = (v0 * B * (io - rho * Gp) + G * Fm * Bp / Q) / D
        zed = (v0 * B * (1 + rho * Ip) - I * Fm * Bp / Q) / D
        assert np.allclose(r.y[0], s0, rtol=1e-13)
        assert np.allclose(r.y[3], v0, rtol=1e-13)
        assert np.allclose(r.y[1], th0 + thd * spec.t_max, rtol=1e-12)
        assert np.allclose(r.y[2], ze0 + zed * spec.t_max, rtol=1e-12)
        if b1 == 0.0:
            assert np.allclose(r.y[2], ze0 + v0 * 5.7 * spec.t_max / 57.0, rtol=1e-12)
            assert np.allclose(r.y[1], th0 + io * v0 * 5.7 * spec.t_max / 57.0, rtol=1e-12)


def _smooth_field():
    """Config-0 harmonics with amplitudes that are cubic polynomials in s: the piecewise-cubic interpolant is
    then one global cubic per harmonic, the field is smooth, and fixed-step RK4 shows its textbook order."""
    fld = W.make_field(0)
    s = np.arange(fld.ns) / (fld.ns - 1)
    amp = fld.bmnc[-1, :].copy()
    fld.bmnc = np.ascontiguousarray(amp[None, :] * (0.2 * s + 0.8 * s ** 2 - 0.3 * s ** 3)[:, None])
    fld.bmnc[:, 0] = W.B00
    return fld


def test_adaptive_trace_matches_brute_force_rk4_smooth_field():
    """(d) classical RK4, fixed tiny step, Richardson ratio ~16, vs the adaptive trace."""
    fld = _smooth_field()
    F = oracle.OracleField(fld)
    P = W.make_particles(0).head(8)
    mu, _ = _mu_for(F, P)
    T = 1e-5
    y_a = F.rk4(M, Q, VREF, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, 4e-9, 2500)
    y_b = F.rk4(M, Q, VREF, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, 2e-9, 5000)
    y_c = F.rk4(M, Q, VREF, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, 1e-9, 10000)
    ratio = np.abs(y_a - y_b).max(axis=1) / np.abs(y_b - y_c).max(axis=1)
    assert np.all(ratio > 11) and np.all(ratio < 23), ratio      # 4th order: ~16
    y_rich = y_c + (y_c - y_b) / 15.0
    spec = W.make_spec(0)
    spec.t_max, spec.rtol, spec.atol = T, 1e-12, 1e-12
    r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    scale = np.array([[1.0], [1.0], [1.0], [VREF]])
    assert (np.abs(r.y - y_rich) / scale).max() < 2e-10


def test_adaptive_trace_matches_brute_force_rk4_config0():
    """(d) on the config-0 field itself.  Its interpolant has slope kinks at the radial nodes, so RK4 converges
    irregularly; the two finest fixed-step runs bracket the answer to ~1e-10 and the adaptive trace at a
    tight tolerance must land inside 1e-9 of them."""
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    P = W.make_particles(0).head(8)
    mu, _ = _mu_for(F, P)
    T = 1e-5
    y_b = F.rk4(M, Q, VREF, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, 5e-10, 20000)
    y_c = F.rk4(M, Q, VREF, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, 2.5e-10, 40000)
    scale = np.array([[1.0], [1.0], [1.0], [VREF]])
    assert (np.abs(y_b - y_c) / scale).max() < 5e-10
    spec = W.make_spec(0)
    spec.t_max, spec.rtol, spec.atol = T, 1e-13, 1e-13
    r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    assert (np.abs(r.y - y_c) / scale).max() < 1e-9


def _axisym_with_modes():
    fld = _smooth_field()            # global cubics in s: no slope kinks, so the invariant is sharp
    keep = fld.xn == 0
    fld.xm, fld.xn, fld.bmnc = fld.xm[keep], fld.xn[keep], np.ascontiguousarray(fld.bmnc[:, keep])
    s = np.arange(fld.ns) / (fld.ns - 1)
    fld.I = 2.0 * s
    fld.mode_m = np.array([3, 4, 6], np.int32)
    fld.mode_n = np.array([2, 2, 2], np.int32)                    # one n, one omega
    fld.mode_omega = np.full(3, 2 * math.pi * 120e3)
    fld.mode_phase = np.array([0.0, 1.0, 2.5])
    env = 4.0 * (s - s ** 3)                                      # cubic envelope, interpolated exactly
    fld.phihat = np.stack([4e4 * env, 3e4 * env, -2e4 * env], axis=1)
    return fld


def test_n_H_minus_omega_P_zeta_invariant_with_modes():
    """(e) axisymmetric equilibrium + modes sharing n and omega: n H - omega P_zeta is exact, while H and
    P_zeta each vary."""
    fld = _axisym_with_modes()
    F = oracle.OracleField(fld)
    chi = lambda s_: fld.psi0 * (0.42 * s_ + 0.05 * s_ * s_)
    P = W.make_particles(0).head(6)
    mu, _ = _mu_for(F, P)
    spec = W.make_spec(0)
    spec.rtol = spec.atol = 1e-11
    spec.t_max = 5e-5
    r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, traj_capacity=40000)
    n, om = 2.0, fld.mode_omega[0]
    seen_variation = 0.0
    for i in range(P.n):
        tr = _traj_arrays(r, i)
        tr = tr[np.linspace(0, len(tr) - 1, 50).astype(int)]
        pz = _p_zeta(F, fld, tr, mu[i], chi)
        H = np.array([0.5 * M * (u * VREF) ** 2 + mu[i] * F.eval_B(s, th, ze)[0]
                      + Q * F.eval_pert(s, th, ze, t)[0] for (t, s, th, ze, u) in tr])
        inv = n * H - om * pz
        ref = abs(n * H[0]) + abs(om * pz[0])
        assert np.abs(inv - inv[0]).max() < 2e-10 * ref
        seen_variation = max(seen_variation, np.abs(H / H[0] - 1).max())
    assert seen_variation > 1e-5


def test_zero_amplitude_modes_reproduce_static_result_bit_for_bit():
    fld0 = W.make_field(0)
    fld1 = W.make_field(0)
    fld1.mode_m = np.array([3], np.int32); fld1.mode_n = np.array([2], np.int32)
    fld1.mode_omega = np.array([7e5]); fld1.mode_phase = np.array([0.3])
    fld1.phihat = np.zeros((fld1.ns, 1))
    F0, F1 = oracle.OracleField(fld0), oracle.OracleField(fld1)
    P = W.make_particles(0).head(8)
    mu, _ = _mu_for(F0, P)
    spec = W.make_spec(0); spec.t_max = 2e-5
    r0 = F0.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    r1 = F1.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    assert np.array_equal(r0.y, r1.y) and np.array_equal(r0.n_acc, r1.n_acc)
