"""Pins for NEXT-4 of SURVEY.md section 8(f) in the oracle: sin (non-stellarator-symmetric) harmonics of B and the
covariant radial component K (field model of PAPER.md:44 without the two simplifications of reading A4).  CPU only.

What fixes the arithmetic: an independent vectorised numpy series and finite differences (the series), a phase-shift
identity (a pure sin harmonic is the cos harmonic shifted by a quarter period), the Euler-Lagrange equations of the
guiding-centre Lagrangian WITH the K term solved numerically (the right-hand side), the identity
K psidot + I thetadot + G zetadot = v_par B that the v_par row of those equations states, energy conservation along a
trace, and the reduction to the closed form O4 when K = 0."""
import dataclasses
import math

import numpy as np
import pytest

import oracle
from paper_2605_16734_b200 import workloads as W

M, Q, VREF = W.ALPHA_MASS, W.ALPHA_CHARGE, W.V_ALPHA


def _asym_field(with_K=True, with_modes=False, ns=41, seed=11):
    """Config-0 recipe at M = N = 4 with non-trivial G, I, iota plus seeded sin harmonics (a few per cent of B00,
    vanishing on the axis like s^{m/2}) and a K of the size I / a^2."""
    fld = W.make_equilibrium(4, 4, ns)
    s = np.arange(ns) / (ns - 1)
    fld.G = 57.0 + 6.0 * s - 2.0 * s ** 2
    fld.I = 4.0 * s + 1.0 * s ** 2
    fld.iota = 0.42 + 0.3 * s
    rng = np.random.default_rng(seed)
    damp = np.exp(-(fld.xm + np.abs(fld.xn)) / 3.0)
    shape = np.power(s[:, None], np.maximum(fld.xm, 1)[None, :] / 2.0)
    fld.bmns = 0.04 * W.B00 * rng.standard_normal(fld.nh)[None, :] * damp[None, :] * shape
    fld.bmns[:, (fld.xm == 0) & (fld.xn == 0)] = 0.0                      # sin(0) carries nothing
    if with_K:
        fld.kmns = 1.5 * rng.standard_normal(fld.nh)[None, :] * damp[None, :] * shape * (1.0 + s[:, None])
        fld.kmnc = 0.7 * rng.standard_normal(fld.nh)[None, :] * damp[None, :] * shape
    if with_modes:
        fld.mode_m = np.array([3, 2], np.int32)
        fld.mode_n = np.array([2, -1], np.int32)
        fld.mode_omega = np.array([7.5e5, -4.0e5])
        fld.mode_phase = np.array([0.3, 2.0])
        env = np.exp(-((s - 0.45) ** 2) / (2 * 0.2 ** 2))
        fld.phihat = np.stack([3e5 * env, 1e5 * env ** 2], axis=1)
    return fld


def _numpy_series(fld, tabc, tabs, s, th, ze):
    """Independent evaluation: polynomial through the 4 stencil nodes by numpy.polyfit, vectorised trig."""
    ns = fld.ns
    u = s * (ns - 1)
    i0 = int(min(max(math.floor(u) - 1, 0), ns - 4))
    nodes = (i0 + np.arange(4)) / (ns - 1)
    ang = fld.xm * th - fld.xn * fld.nfp * ze
    X = Xs = Xth = Xze = 0.0
    for tab, f0, f1 in ((tabc, np.cos, lambda a: -np.sin(a)), (tabs, np.sin, np.cos)):
        if tab is None:
            continue
        coef = np.polyfit(nodes - s, tab[i0:i0 + 4], 3)                  # [4][nh], value and slope at s
        b, bs = coef[3], coef[2]
        X += np.sum(b * f0(ang))
        Xs += np.sum(bs * f0(ang))
        Xth += np.sum(fld.xm * b * f1(ang))
        Xze += np.sum(-fld.xn * fld.nfp * b * f1(ang))
    return np.array([X, Xs, Xth, Xze])


def test_sin_harmonics_and_K_series_against_numpy_and_finite_differences():
    fld = _asym_field()
    F = oracle.OracleField(fld)
    rng = np.random.default_rng(3)
    for _ in range(8):
        s, th, ze = rng.uniform(0.05, 0.95), rng.uniform(-4, 4), rng.uniform(-4, 4)
        got = F.eval_B(s, th, ze)
        ref = _numpy_series(fld, fld.bmnc, fld.bmns, s, th, ze)
        assert np.allclose(got, ref, rtol=1e-10, atol=1e-10 * 5.7 * np.array([1, 40, 1, 1]))
        gk = F.eval_K(s, th, ze)
        rk = _numpy_series(fld, fld.kmnc, fld.kmns, s, th, ze)
        assert np.allclose(gk, rk, rtol=1e-10, atol=1e-10 * np.array([1, 40, 1, 1]))
        # the sin tables matter here, else the comparison pins nothing
        assert abs(got[0] - _numpy_series(fld, fld.bmnc, None, s, th, ze)[0]) > 1e-4
        # derivatives in theta and zeta by central differences (the series is smooth in the angles)
        h = 1e-5
        for ev in (F.eval_B, F.eval_K):
            v = ev(s, th, ze)
            dth = (ev(s, th + h, ze)[0] - ev(s, th - h, ze)[0]) / (2 * h)
            dze = (ev(s, th, ze + h)[0] - ev(s, th, ze - h)[0]) / (2 * h)
            # truncation of the difference quotient: h^2 (n nfp)^3 / 6 ~ 1e-7; a wrong sign or factor is O(1)
            assert abs(dth - v[2]) < 1e-6 * max(1.0, abs(v[2])) and abs(dze - v[3]) < 1e-6 * max(1.0, abs(v[3]))
    # inside one radial cell the interpolant is a cubic: the s-derivative by central differences
    s = (10 + 0.4) / (fld.ns - 1)
    for ev in (F.eval_B, F.eval_K):
        h = 1e-6
        ds = (ev(s + h, 0.3, 0.2)[0] - ev(s - h, 0.3, 0.2)[0]) / (2 * h)
        assert abs(ds - ev(s, 0.3, 0.2)[1]) < 1e-7 * max(1.0, abs(ds))


def test_pure_sin_harmonic_is_the_cos_harmonic_shifted_by_a_quarter_period():
    """b sin(m theta - n nfp zeta) = b cos(m (theta - pi / 2m) - n nfp zeta): a field whose only angle-dependent
    harmonic is a sin term equals the matching cos field evaluated at theta - pi / (2 m), value and derivatives."""
    ns = 21
    s_n = np.arange(ns) / (ns - 1)
    xm, xn = np.array([0, 3], np.int32), np.array([0, 2], np.int32)
    amp = 0.3 * s_n ** 1.5
    zero = np.zeros(ns)
    base = dict(ns=ns, nfp=4, xm=xm, xn=xn, G=np.full(ns, 57.0), I=np.zeros(ns), iota=np.full(ns, 0.5), psi0=W.PSI0)
    cosf = W.Field(bmnc=np.stack([np.full(ns, 5.7), amp], axis=1), **base)
    sinf = W.Field(bmnc=np.stack([np.full(ns, 5.7), zero], axis=1), bmns=np.stack([zero, amp], axis=1), **base)
    Fc, Fs = oracle.OracleField(cosf), oracle.OracleField(sinf)
    for s, th, ze in ((0.33, 0.7, -1.1), (0.81, -2.0, 0.4)):
        a = Fs.eval_B(s, th, ze)
        b = Fc.eval_B(s, th - math.pi / 6.0, ze)
        assert np.allclose(a, b, rtol=1e-13, atol=1e-14)
        assert abs(a[2]) > 1e-3 and abs(a[3]) > 1e-3


def _lagrangian_rhs_with_K(F, fld, mu, t, z):
    """Solve sum_j omega_ij zdot_j = dH/dz_i + dLambda_i/dt, omega_ij = dLambda_j/dz_i - dLambda_i/dz_j for
      L = Lambda_psi psidot + Lambda_theta thetadot + Lambda_zeta zetadot - H,
      Lambda_psi = q rho_c K, Lambda_theta = q (psi + rho_c I), Lambda_zeta = q (rho_c G - chi), chi' = iota,
    with every derivative by Richardson-extrapolated central differences of the oracle's POINT evaluations
    (eval_B, eval_K, eval_profiles, eval_pert): nothing of oracle_rhs_general's algebra is used."""
    psi0 = fld.psi0

    def parts(zz, tt):
        s, th, ze, v = zz
        B = F.eval_B(s, th, ze)[0]
        K = F.eval_K(s, th, ze)[0]
        G, _, I, _, _, _ = F.eval_profiles(s)
        pt = F.eval_pert(s, th, ze, tt)
        rho_c = M * v / (Q * B) + pt[4]
        return np.array([Q * rho_c * K, Q * (psi0 * s + rho_c * I), Q * rho_c * G,
                         0.5 * M * v * v + mu * B + Q * pt[0]])

    steps = np.array([2e-4, 1e-3, 1e-3, 2e-3 * VREF])

    def rich(fn, h):
        cd = lambda hh: (fn(hh) - fn(-hh)) / (2 * hh)
        return (4.0 * cd(h / 2) - cd(h)) / 3.0

    D = np.array([rich(lambda hh, i=i: parts(z + hh * np.eye(4)[i], t), steps[i]) for i in range(4)])
    Dt = rich(lambda hh: parts(z, t + hh), 2e-8)
    D[0, :3] /= psi0                                                   # d/ds -> d/dpsi
    iota = F.eval_profiles(z[0])[4]
    Lam = np.zeros((4, 4))                                             # Lam[j][i] = dLambda_j / dz_i
    Lam[0], Lam[1], Lam[2] = D[:, 0], D[:, 1], D[:, 2]
    Lam[0, 0] = 0.0                                                    # cancels in omega; avoid its psi0 mismatch
    Lam[2, 0] -= Q * iota
    omega = Lam.T - Lam
    dH = D[:, 3].copy()
    dH[0] /= psi0
    rhs = dH + np.array([Dt[0], Dt[1], Dt[2], 0.0])
    scale = np.abs(omega).max(axis=1, keepdims=True)
    zd = np.linalg.solve(omega / scale, rhs / scale[:, 0])
    zd[0] /= psi0                                                      # psidot -> sdot
    return zd


@pytest.mark.parametrize("with_modes", [False, True])
def test_general_rhs_equals_euler_lagrange_equations_with_K(with_modes):
    fld = _asym_field(with_K=True, with_modes=with_modes)
    F = oracle.OracleField(fld)
    F0 = oracle.OracleField(dataclasses.replace(fld, kmnc=None, kmns=None))
    rng = np.random.default_rng(5)
    moved = 0.0
    for _ in range(6):
        s = (math.floor(rng.uniform(0.15, 0.85) * (fld.ns - 1)) + 0.5) / (fld.ns - 1)
        th, ze = rng.uniform(-3, 3, 2)
        v = rng.uniform(0.2, 1.0) * VREF * rng.choice([-1, 1])
        B = F.eval_B(s, th, ze)[0]
        mu = 0.5 * M * (VREF ** 2 - v ** 2) / B
        t = float(rng.uniform(0, 1e-5))
        got = F.rhs(M, Q, mu, VREF, t, [s, th, ze, v / VREF]) * np.array([1, 1, 1, VREF])
        ref = _lagrangian_rhs_with_K(F, fld, mu, t, np.array([s, th, ze, v]))
        tol = 2e-6 * np.maximum(np.abs(ref), np.array([1e-2 * abs(ref[1]), 0, 0, 1e-3 * abs(ref[3]) + 1.0]))
        assert np.all(np.abs(got - ref) <= tol + 1e-7 * np.abs(ref)), (got, ref)
        # the v_par row of the equations, by hand: K psidot + I thetadot + G zetadot = v_par B
        K = F.eval_K(s, th, ze)[0]
        G, _, I, _, _, _ = F.eval_profiles(s)
        lhs = K * got[0] * fld.psi0 + I * got[1] + G * got[2]
        assert abs(lhs - v * B) < 1e-12 * abs(v * B)
        base = F0.rhs(M, Q, mu, VREF, t, [s, th, ze, v / VREF]) * np.array([1, 1, 1, VREF])
        moved = max(moved, abs(got[0] - base[0]) / abs(base[0]))
    assert moved > 1e-2                                                 # K matters in this test


def test_general_form_reduces_to_the_closed_form_without_K():
    fld = _asym_field(with_K=False, with_modes=True)
    F = oracle.OracleField(fld)
    rng = np.random.default_rng(9)
    for _ in range(10):
        y = [rng.uniform(0.05, 0.95), rng.uniform(-3, 3), rng.uniform(-3, 3), rng.uniform(-1, 1)]
        mu = rng.uniform(0.0, 1.0) * 0.5 * M * VREF ** 2 / 5.7
        a = F.rhs(M, Q, mu, VREF, 3e-6, y)
        b = F.rhs_general(M, Q, mu, VREF, 3e-6, y)
        assert np.allclose(a, b, rtol=1e-11, atol=1e-11 * np.abs(a).max())


def test_energy_conserved_with_sin_harmonics_and_K():
    """A time-independent field conserves E = m v^2 / 2 + mu B whatever K and the symmetry of B (the system is
    antisymmetric): drift bounded by the tolerance and shrinking with it."""
    fld = _asym_field(with_K=True)
    F = oracle.OracleField(fld)
    P = W.make_particles(0).head(8)
    B0 = F.eval_B_many(P.s, P.theta, P.zeta)[:, 0]
    mu = W.mu_from(P, B0)
    E0 = 0.5 * M * P.vpar ** 2 + mu * B0
    drift = []
    for rtol in (1e-7, 1e-9):
        spec = W.make_spec(0)
        spec.rtol = spec.atol = rtol
        spec.t_max = 2e-5
        r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
        assert (r.status == 0).all()
        B1 = F.eval_B_many(r.y[0], r.y[1], r.y[2])[:, 0]
        E1 = 0.5 * M * r.y[3] ** 2 + mu * B1
        drift.append(np.abs(E1 / E0 - 1).max())
        assert np.abs(r.y[0] - P.s).max() > 1e-3                        # the orbits do move radially
    assert drift[0] < 1e-5 and drift[1] < 1e-7 and drift[1] < 0.1 * drift[0]
