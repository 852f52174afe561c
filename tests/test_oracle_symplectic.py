"""Pins for NEXT-3 of SURVEY.md section 8(f) in the oracle: the symplectic explicit-implicit Euler integrator for
non-canonical guiding-centre orbits ("uses the explicit-implicit Euler scheme of (Albert et al., 2020)";
PAPER.md:60-62 and Fig. 1 left: "the symplectic algorithm exhibits a stable moving time average of the energy";
reading A28 of DESIGN.md).  CPU only.

What fixes the arithmetic, none of it the oracle's own formulas re-typed:
  * the textbook symplectic Euler map  p' = p - h dK/dq(q, p'),  q' = q + h dK/dp(q, p')  built independently in
    canonical variables (theta, zeta, p_theta, p_zeta), with K evaluated from the oracle's POINT evaluations of B and
    the profiles, s(p_theta, p_zeta) found by a scipy root solve and every derivative of K taken by finite
    differences -- pins the chain rule through s, all partial derivatives and the explicit/implicit split;
  * the symplectic condition M^T J M = J of the one-step map, differentiated numerically, which the explicit Euler
    map of the same equations violates at O(h);
  * convergence to the Dormand-Prince orbit (itself pinned to the Euler-Lagrange equations) at first order in h;
  * invariants: in a field with only n = 0 harmonics p_zeta is conserved to rounding (equation (2) has no force
    term), in a field with B00 only every step is the exact closed-form orbit;
  * the behaviour the paper shows: bounded energy error without drift, against the drift of Dormand-Prince.
"""
import math

import numpy as np
import pytest
from scipy.optimize import brentq, fsolve

import oracle
from paper_2605_16734_b200 import workloads as W

M, Q, VREF = W.ALPHA_MASS, W.ALPHA_CHARGE, W.V_ALPHA


def _field_I():
    """Static field with I != 0, G' != 0 and a quadratic chi (exact under cubic interpolation)."""
    fld = W.make_equilibrium(4, 3, 41)
    s = np.arange(fld.ns) / (fld.ns - 1)
    fld.G = 57.0 + 3.0 * s - 1.0 * s ** 2
    fld.I = 3.0 * s + 1.0 * s ** 2
    fld.iota = 0.42 + 0.3 * s
    chi = fld.psi0 * (0.42 * s + 0.15 * s ** 2)
    return fld, chi


def _chi0(fld):
    s = np.arange(fld.ns) / (fld.ns - 1)
    return fld.psi0 * (0.42 * s + 0.05 * s ** 2)            # iota = 0.42 + 0.1 s of the BASELINE recipes


def _canon_funcs(F, fld, chi_nodes, mu):
    """p_theta(s, p_zeta) and H(s, theta, zeta, p_zeta) from point evaluations (definitions of the canonical momenta
    and of the energy, not of the scheme)."""
    s_n = np.arange(fld.ns) / (fld.ns - 1)

    def chi(s):                                         # chi is a polynomial of degree <= 3 in these tests
        return np.polyval(np.polyfit(s_n, chi_nodes, 3), s)

    def rho(s, pz):
        G = F.eval_profiles(s)[0]
        return (pz / Q + chi(s)) / G

    def ptheta(s, pz):
        I = F.eval_profiles(s)[2]
        return Q * (fld.psi0 * s + rho(s, pz) * I)

    def H(s, th, ze, pz):
        B = F.eval_B(s, th, ze)[0]
        return (Q * rho(s, pz) * B) ** 2 / (2 * M) + mu * B

    def s_of(pth, pz, guess):
        return brentq(lambda s: ptheta(s, pz) - pth, guess - 0.05, guess + 0.05, xtol=1e-15, rtol=1e-15)

    def K(th, ze, pth, pz, guess):
        return H(s_of(pth, pz, guess), th, ze, pz)
    return ptheta, H, s_of, K


def test_one_step_is_the_textbook_symplectic_euler_map_in_canonical_variables():
    fld, chi = _field_I()
    F = oracle.OracleField(fld)
    s0, th0, ze0, v0 = 0.37, 1.3, 0.4, 0.6 * VREF
    B0 = F.eval_B(s0, th0, ze0)[0]
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / B0
    pz0 = F.symplectic_pzeta(M, Q, chi, s0, th0, ze0, v0)
    ptheta, H, s_of, K = _canon_funcs(F, fld, chi, mu)
    pth0 = ptheta(s0, pz0)
    h = 4e-8
    z1, it = F.symplectic_step(M, Q, mu, chi, h, [s0, th0, ze0, pz0])
    assert 2 <= it <= 8
    # independent construction: unknowns p' = (p_theta', p_zeta'), scaled by q psi0
    unit = Q * fld.psi0
    e_ang, e_p = 1e-5, 1e-5 * unit

    def dK_dq(pth, pz):
        a = (K(th0 + e_ang, ze0, pth, pz, s0) - K(th0 - e_ang, ze0, pth, pz, s0)) / (2 * e_ang)
        b = (K(th0, ze0 + e_ang, pth, pz, s0) - K(th0, ze0 - e_ang, pth, pz, s0)) / (2 * e_ang)
        return a, b

    def dK_dp(pth, pz):
        a = (K(th0, ze0, pth + e_p, pz, s0) - K(th0, ze0, pth - e_p, pz, s0)) / (2 * e_p)
        b = (K(th0, ze0, pth, pz + e_p, s0) - K(th0, ze0, pth, pz - e_p, s0)) / (2 * e_p)
        return a, b

    def resid(x):
        pth, pz = x[0] * unit, x[1] * unit
        a, b = dK_dq(pth, pz)
        return [(pth - pth0 + h * a) / unit, (pz - pz0 + h * b) / unit]

    x = fsolve(resid, [pth0 / unit, pz0 / unit], xtol=1e-15)
    pth1, pz1 = x[0] * unit, x[1] * unit
    a, b = dK_dp(pth1, pz1)
    th1, ze1 = th0 + h * a, ze0 + h * b
    s1 = s_of(pth1, pz1, s0)
    # increments agree to the accuracy of the finite differences (1e-6 relative), far below any algebra mistake
    assert abs((z1[0] - s0) - (s1 - s0)) < 2e-6 * abs(s1 - s0)
    assert abs((z1[1] - th0) - (th1 - th0)) < 2e-6 * abs(th1 - th0)
    assert abs((z1[2] - ze0) - (ze1 - ze0)) < 2e-6 * abs(ze1 - ze0)
    assert abs((z1[3] - pz0) - (pz1 - pz0)) < 2e-6 * abs(pz1 - pz0)
    assert abs(s1 - s0) > 1e-7 and abs(pz1 - pz0) > 1e-9 * abs(pz0)     # the step really moves every component


def _map_jacobian(F, fld, chi, mu, h, z0, step):
    """d(theta', zeta', p_theta', p_zeta') / d(theta, zeta, p_theta, p_zeta) of `step` by central differences, momenta
    in units of q psi0."""
    ptheta, H, s_of, K = _canon_funcs(F, fld, chi, mu)
    unit = Q * fld.psi0

    def to_canon(z):
        return np.array([z[1], z[2], ptheta(z[0], z[3]) / unit, z[3] / unit])

    def from_canon(c, guess):
        pz = c[3] * unit
        return np.array([s_of(c[2] * unit, pz, guess), c[0], c[1], pz])

    c0 = to_canon(z0)
    Mx = np.zeros((4, 4))
    for j in range(4):
        e = np.zeros(4)
        e[j] = 1e-5
        zp = step(from_canon(c0 + e, z0[0]))
        zm = step(from_canon(c0 - e, z0[0]))
        Mx[:, j] = (to_canon(zp) - to_canon(zm)) / 2e-5
    return Mx


def test_one_step_map_is_symplectic_and_explicit_euler_is_not():
    fld, chi = _field_I()
    F = oracle.OracleField(fld)
    s0, th0, ze0, v0 = 0.42, 2.1, -0.3, -0.45 * VREF
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / F.eval_B(s0, th0, ze0)[0]
    z0 = np.array([s0, th0, ze0, F.symplectic_pzeta(M, Q, chi, s0, th0, ze0, v0)])
    h = 1e-7
    J = np.array([[0, 0, 1, 0], [0, 0, 0, 1], [-1, 0, 0, 0], [0, -1, 0, 0]], float)

    def sym(z):
        return F.symplectic_step(M, Q, mu, chi, h, z)[0]

    def explicit_euler(z):
        v = F.symplectic_vpar(M, Q, chi, z[0], z[1], z[2], z[3])
        d = F.rhs(M, Q, mu, 1.0, 0.0, [z[0], z[1], z[2], v])
        s1, th1, ze1, v1 = z[0] + h * d[0], z[1] + h * d[1], z[2] + h * d[2], v + h * d[3]
        return np.array([s1, th1, ze1, F.symplectic_pzeta(M, Q, chi, s1, th1, ze1, v1)])

    Ms = _map_jacobian(F, fld, chi, mu, h, z0, sym)
    Me = _map_jacobian(F, fld, chi, mu, h, z0, explicit_euler)
    defect_s = np.abs(Ms.T @ J @ Ms - J).max()
    defect_e = np.abs(Me.T @ J @ Me - J).max()
    assert np.abs(Ms - np.eye(4)).max() > 1e-3          # not the identity: the test has something to see
    assert defect_s < 2e-8                              # finite-difference noise
    assert defect_e > 100 * defect_s and defect_e > 1e-6


def test_first_order_convergence_to_the_dormand_prince_orbit():
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    chi = _chi0(fld)
    P = W.make_particles(0).head(12)
    mu = W.mu_from(P, F.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    spec = W.make_spec(0)
    spec.rtol = spec.atol = 1e-12
    T = 4e-6
    ref = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=T).y
    err = {}
    for n in (1000, 2000, 4000):
        r = F.trace_symplectic(M, Q, P.s, P.theta, P.zeta, P.vpar, mu, chi, dt=T / n, nsteps=n)
        assert (r.status == 0).all() and (r.n_steps == n).all() and np.allclose(r.t, T, rtol=1e-12)
        err[n] = np.abs(r.y - ref).max(axis=1) / np.array([1.0, 1.0, 1.0, VREF])
    for c in range(4):
        assert 1.8 < err[1000][c] / err[2000][c] < 2.2, (c, err)
        assert 1.8 < err[2000][c] / err[4000][c] < 2.2, (c, err)
    assert err[4000].max() < 5e-3


def test_p_zeta_exact_in_axisymmetric_field_and_closed_form_orbit_in_B00_field():
    # (i) n = 0 harmonics only: dH/dzeta = 0, so equation (2) keeps p_zeta to the last bit whatever the step
    fld = W.make_field(0)
    keep = fld.xn == 0
    fld.xm, fld.xn, fld.bmnc = fld.xm[keep], fld.xn[keep], np.ascontiguousarray(fld.bmnc[:, keep])
    F = oracle.OracleField(fld)
    chi = _chi0(fld)
    P = W.make_particles(0).head(6)
    mu = W.mu_from(P, F.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    r = F.trace_symplectic(M, Q, P.s, P.theta, P.zeta, P.vpar, mu, chi, dt=5e-8, nsteps=400)
    assert (r.status == 0).all()
    for i in range(P.n):
        p0 = F.symplectic_pzeta(M, Q, chi, P.s[i], P.theta[i], P.zeta[i], P.vpar[i])
        p1 = F.symplectic_pzeta(M, Q, chi, *r.y[:, i])
        assert abs(p1 / p0 - 1.0) < 1e-13
        assert abs(r.y[0, i] - P.s[i]) > 1e-4           # while s moved
    # (ii) only B00, constant G, I = 0: dH/dtheta = dH/dzeta = 0, momenta and s are constant and (3), (4) are the
    # exact rates zeta' = v B / G, theta' = iota zeta' (closed form of test_oracle_physics), for any h
    ns = 21
    s_n = np.arange(ns) / (ns - 1)
    fld = W.Field(ns=ns, nfp=4, xm=np.zeros(1, np.int32), xn=np.zeros(1, np.int32), bmnc=np.full((ns, 1), 5.7),
                  G=np.full(ns, 57.0), I=np.zeros(ns), iota=0.42 + 0.1 * s_n, psi0=W.PSI0)
    F = oracle.OracleField(fld)
    chi = _chi0(fld)
    s0 = np.array([0.3, 0.6]); th0 = np.array([0.5, 1.0]); ze0 = np.array([0.1, -2.0])
    v0 = np.array([0.8, -0.5]) * VREF
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / 5.7
    r = F.trace_symplectic(M, Q, s0, th0, ze0, v0, mu, chi, dt=2e-7, nsteps=100)
    T = 2e-5
    assert np.allclose(r.y[0], s0, rtol=1e-13) and np.allclose(r.y[3], v0, rtol=1e-12)
    assert np.allclose(r.y[2], ze0 + v0 * 5.7 * T / 57.0, rtol=1e-12)
    assert np.allclose(r.y[1], th0 + (0.42 + 0.1 * s0) * v0 * 5.7 * T / 57.0, rtol=1e-12)


def _energy(F, y, mu):
    B = F.eval_B_many(y[0], y[1], y[2])[:, 0]
    return 0.5 * M * y[3] ** 2 + mu * B


def test_energy_moving_average_is_stable_while_dormand_prince_drifts():
    """PAPER.md:60-62 / Fig. 1 left on a smooth field (cubic-in-s amplitudes: no kinks at the radial nodes)."""
    fld = W.make_field(0)
    s = np.arange(fld.ns) / (fld.ns - 1)
    amp = fld.bmnc[-1, :].copy()
    fld.bmnc = np.ascontiguousarray(amp[None, :] * (0.2 * s + 0.8 * s ** 2 - 0.3 * s ** 3)[:, None])
    fld.bmnc[:, 0] = W.B00
    F = oracle.OracleField(fld)
    chi = _chi0(fld)
    P = W.make_particles(0).head(4)
    mu = W.mu_from(P, F.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    E0 = _energy(F, np.stack([P.s, P.theta, P.zeta, P.vpar]), mu)
    dt, nsteps, stride = 2.5e-8, 16000, 20                   # 4e-4 s
    r = F.trace_symplectic(M, Q, P.s, P.theta, P.zeta, P.vpar, mu, chi, dt=dt, nsteps=nsteps,
                           sample_stride=stride, nsamp=nsteps // stride + 1)
    assert (r.status == 0).all() and (r.sample_end == nsteps // stride + 1).all()
    spec = W.make_spec(0)
    spec.rtol = spec.atol = 1e-6                             # a Runge-Kutta run of comparable cost
    d = F.trace_sampled(spec, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, dt * stride, nsteps // stride + 1,
                        t_max=dt * nsteps)
    for i in range(P.n):
        es = _energy(F, r.samples[:, :, i], mu[i]) / E0[i] - 1.0
        ed = _energy(F, d.samples[:, :, i], mu[i]) / E0[i] - 1.0
        w = len(es) // 4
        first, last = es[:w].mean(), es[-w:].mean()
        amp_s = es.max() - es.min()
        assert amp_s < 2e-2                                   # bounded, O(h)
        assert abs(last - first) < 0.01 * amp_s               # the moving average does not drift
        # Dormand-Prince: a net drift larger than its own fluctuation around it
        assert abs(ed[-w:].mean() - ed[:w].mean()) > 4 * abs(last - first)


def test_stop_rules_status_and_samples_layout():
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    chi = _chi0(fld)
    P = W.make_particles(0).head(8)
    mu = W.mu_from(P, F.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    # a loss surface just outside the start radius: a particle that drifts outward is stopped at the END of the
    # step that crosses it (O7), with t_out = t0 + steps * dt and its later samples untouched
    r = F.trace_symplectic(M, Q, P.s, P.theta, P.zeta, P.vpar, mu, chi, dt=5e-9, nsteps=600, t0=1e-6, s_loss=0.2502,
                           s_min=0.2498, sample_stride=100, nsamp=7)
    assert set(r.status) <= {0, 1, 2} and (r.status == 1).any() and (r.status == 2).any()
    for i in range(P.n):
        assert math.isclose(r.t[i], 1e-6 + r.n_steps[i] * 5e-9, rel_tol=1e-14)
        if r.status[i] == 1:
            assert r.y[0, i] >= 0.2502 and r.n_steps[i] < 600
        if r.status[i] == 2:
            assert r.y[0, i] <= 0.2498 and r.n_steps[i] < 600
        assert r.sample_end[i] == 1 + r.n_steps[i] // 100
        assert np.isfinite(r.samples[:, :r.sample_end[i], i]).all()
        assert np.isnan(r.samples[:, r.sample_end[i]:, i]).all()
        assert np.array_equal(r.samples[:3, 0, i], [P.s[i], P.theta[i], P.zeta[i]])
    # the stopped particle equals the same particle run for exactly n_steps steps without the stop rule
    i = int(np.nonzero(r.status == 1)[0][0])
    q = F.trace_symplectic(M, Q, P.s[i:i + 1], P.theta[i:i + 1], P.zeta[i:i + 1], P.vpar[i:i + 1], mu[i:i + 1], chi,
                           dt=5e-9, nsteps=int(r.n_steps[i]), t0=1e-6)
    assert np.array_equal(q.y[:, 0], r.y[:, i])
    # non-finite input -> status 4, no steps; modes or K tables are refused
    bad = F.trace_symplectic(M, Q, [float("nan")], [0.0], [0.0], [1e6], [1e-14], chi, dt=5e-9, nsteps=5)
    assert bad.status[0] == 4 and bad.n_steps[0] == 0
    with pytest.raises(ValueError):
        oracle.OracleField(W.make_field(2)).trace_symplectic(M, Q, P.s, P.theta, P.zeta, P.vpar, mu, chi, dt=5e-9,
                                                             nsteps=5)
