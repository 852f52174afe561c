"""Pins for the oracle's radial interpolation (O1) and harmonic sums (O2, O3).  CPU only.

Each pin goes around the oracle's own formulae: polynomial exactness, numpy library routines on the
same four nodes, finite differences, an independent vectorised numpy series, and closed forms.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2605_16734_b200 import workloads as W


@pytest.mark.parametrize("ns", [4, 16, 51, 101])
def test_lagrange_partition_and_cubic_exactness(ns):
    rng = np.random.default_rng(1)
    coef = rng.standard_normal(4)
    poly = np.polynomial.Polynomial(coef)
    nodes = np.arange(ns) / (ns - 1)
    for s in np.concatenate([rng.uniform(0, 1, 40), [0.0, 1.0, 0.5, 1.0 / (ns - 1)]]):
        i0, w, dw = oracle.lagrange(ns, float(s))
        assert 0 <= i0 <= ns - 4
        assert abs(w.sum() - 1.0) < 1e-13
        assert abs(dw.sum()) < 1e-10 * ns
        vals = poly(nodes[i0:i0 + 4])
        assert abs(w @ vals - poly(s)) < 1e-12 * (1 + abs(poly(s)))
        assert abs(dw @ vals - poly.deriv()(s)) < 1e-10 * (1 + abs(poly.deriv()(s))) * ns


def test_lagrange_stencil_choice_and_edges():
    ns = 51
    # interior: the query lies in the middle interval of the stencil (x in [1,2])
    for s in (0.25, 0.251, 0.5, 0.73):
        i0, w, _ = oracle.lagrange(ns, s)
        x = s * (ns - 1) - i0
        assert 1.0 <= x < 2.0 + 1e-12
        assert i0 == min(max(math.floor(s * (ns - 1)) - 1, 0), ns - 4)
    # clamped ends and extrapolation outside [0,1] (A6)
    assert oracle.lagrange(ns, 0.0)[0] == 0
    assert oracle.lagrange(ns, 0.001)[0] == 0
    assert oracle.lagrange(ns, -0.3)[0] == 0
    assert oracle.lagrange(ns, 1.0)[0] == ns - 4
    assert oracle.lagrange(ns, 0.999)[0] == ns - 4
    assert oracle.lagrange(ns, 1.7)[0] == ns - 4
    assert oracle.lagrange(ns, float("nan"))[0] == 0
    # at a node the weights are a Kronecker delta
    i0, w, _ = oracle.lagrange(ns, 10 / (ns - 1))
    j = 10 - i0
    e = np.zeros(4)
    e[j] = 1.0
    assert np.allclose(w, e, atol=1e-12)


def test_lagrange_matches_numpy_polyfit_interpolating_polynomial():
    ns = 33
    rng = np.random.default_rng(2)
    tab = rng.standard_normal(ns)
    nodes = np.arange(ns) / (ns - 1)
    for s in rng.uniform(-0.02, 1.02, 25):
        i0, w, dw = oracle.lagrange(ns, float(s))
        P = np.poly1d(np.polyfit(nodes[i0:i0 + 4] - nodes[i0], tab[i0:i0 + 4], 3))   # library routine
        assert abs(w @ tab[i0:i0 + 4] - P(s - nodes[i0])) < 1e-10
        assert abs(dw @ tab[i0:i0 + 4] - P.deriv()(s - nodes[i0])) < 1e-8


def _numpy_series(fld, s, th, ze):
    """Independent route: numpy.polyfit through the four stencil nodes, vectorised cos/sin series."""
    ns = fld.ns
    nodes = np.arange(ns) / (ns - 1)
    c = math.floor(s * (ns - 1))
    i0 = min(max(c - 1, 0), ns - 4)
    xs = nodes[i0:i0 + 4] - nodes[i0]
    V = np.vander(xs, 4)
    coef = np.linalg.solve(V, fld.bmnc[i0:i0 + 4, :])            # cubic through the 4 nodes, per harmonic
    x = s - nodes[i0]
    b = coef[0] * x ** 3 + coef[1] * x ** 2 + coef[2] * x + coef[3]
    bs = 3 * coef[0] * x ** 2 + 2 * coef[1] * x + coef[2]
    ang = fld.xm * th - fld.xn * fld.nfp * ze
    return np.array([np.sum(b * np.cos(ang)), np.sum(bs * np.cos(ang)),
                     np.sum(-fld.xm * b * np.sin(ang)), np.sum(fld.xn * fld.nfp * b * np.sin(ang))])


@pytest.mark.parametrize("config", [0, 1])
def test_eval_B_matches_numpy_series_and_finite_differences(config):
    fld = W.make_field(config)
    F = oracle.OracleField(fld)
    rng = np.random.default_rng(3)
    for _ in range(6):
        s = float(rng.uniform(0.05, 0.95))
        # keep s +- d inside one radial cell so that the piecewise cubic is smooth
        u = s * (fld.ns - 1)
        s = (math.floor(u) + 0.5) / (fld.ns - 1)
        th, ze = rng.uniform(-10, 10, 2)
        out = F.eval_B(s, th, ze)
        ref = _numpy_series(fld, s, th, ze)
        assert np.allclose(out, ref, rtol=1e-10, atol=1e-10)
        d = 1e-5
        fd_s = (F.eval_B(s + d, th, ze)[0] - F.eval_B(s - d, th, ze)[0]) / (2 * d)
        fd_t = (F.eval_B(s, th + d, ze)[0] - F.eval_B(s, th - d, ze)[0]) / (2 * d)
        fd_z = (F.eval_B(s, th, ze + d)[0] - F.eval_B(s, th, ze - d)[0]) / (2 * d)
        scale = 1.0 + np.abs(out[1:])
        assert abs(fd_s - out[1]) < 2e-7 * scale[0] * 100
        assert abs(fd_t - out[2]) < 2e-7 * scale[1] * 100
        assert abs(fd_z - out[3]) < 2e-7 * scale[2] * 100


def test_eval_B_single_harmonic_closed_form():
    """B = B00 + b(s) cos(2 theta - 3*nfp*zeta) with b cubic in s: the cubic Lagrange interpolant is exact."""
    ns, nfp = 21, 5
    s_nodes = np.arange(ns) / (ns - 1)
    bfun = lambda s: 0.3 * s ** 3 - 0.2 * s + 0.05
    dbfun = lambda s: 0.9 * s ** 2 - 0.2
    fld = W.Field(ns=ns, nfp=nfp, xm=np.array([0, 2], np.int32), xn=np.array([0, 3], np.int32),
                  bmnc=np.stack([np.full(ns, 2.0), bfun(s_nodes)], axis=1), G=np.full(ns, 10.0),
                  I=np.zeros(ns), iota=np.full(ns, 0.4), psi0=1.0)
    F = oracle.OracleField(fld)
    for s, th, ze in [(0.37, 0.3, 1.1), (0.02, -2.0, 4.0), (0.99, 7.0, -3.0)]:
        ang = 2 * th - 3 * nfp * ze
        out = F.eval_B(s, th, ze)
        exp = [2.0 + bfun(s) * math.cos(ang), dbfun(s) * math.cos(ang),
               -2 * bfun(s) * math.sin(ang), 3 * nfp * bfun(s) * math.sin(ang)]
        assert np.allclose(out, exp, rtol=1e-12, atol=1e-12)


def test_profiles_interpolate_cubics_exactly():
    ns = 31
    s_nodes = np.arange(ns) / (ns - 1)
    fld = W.make_equilibrium(2, 2, ns)
    fld.G = 50 + 3 * s_nodes - s_nodes ** 3
    fld.I = 0.7 * s_nodes ** 2
    fld.iota = 0.42 + 0.1 * s_nodes
    F = oracle.OracleField(fld)
    for s in (0.013, 0.4, 0.77, 0.995):
        G, Gs, I, Is, io, ios = F.eval_profiles(s)
        assert np.allclose([G, Gs, I, Is, io, ios],
                           [50 + 3 * s - s ** 3, 3 - 3 * s ** 2, 0.7 * s ** 2, 1.4 * s, 0.42 + 0.1 * s, 0.1],
                           rtol=1e-11, atol=1e-11)


def _pert_field():
    fld = W.make_equilibrium(4, 4, 41)
    s = np.arange(fld.ns) / (fld.ns - 1)
    fld.G = 57.0 + 2.0 * s
    fld.I = 1.5 * s
    fld.mode_m = np.array([3, 5, 2], np.int32)
    fld.mode_n = np.array([2, 2, -1], np.int32)
    fld.mode_omega = np.array([7.5e5, 7.5e5, -4.0e5])
    fld.mode_phase = np.array([0.0, 0.7, 2.0])
    env = np.exp(-((s - 0.45) ** 2) / (2 * 0.15 ** 2))
    fld.phihat = np.stack([3e3 * env, -2e3 * env * (1 + s), 1e3 * env ** 2], axis=1)
    return fld


def test_pert_derivatives_by_finite_differences():
    fld = _pert_field()
    F = oracle.OracleField(fld)
    rng = np.random.default_rng(4)
    for _ in range(5):
        s = (math.floor(rng.uniform(0.1, 0.9) * (fld.ns - 1)) + 0.5) / (fld.ns - 1)
        th, ze = rng.uniform(-6, 6, 2)
        t = float(rng.uniform(0, 1e-4))
        o = F.eval_pert(s, th, ze, t)
        d, dt = 1e-5, 1e-10
        fd = lambda i, a, b, h: (F.eval_pert(*a)[i] - F.eval_pert(*b)[i]) / (2 * h)
        Phi_s = fd(0, (s + d, th, ze, t), (s - d, th, ze, t), d)
        Phi_t = fd(0, (s, th + d, ze, t), (s, th - d, ze, t), d)
        Phi_z = fd(0, (s, th, ze + d, t), (s, th, ze - d, t), d)
        al_s = fd(4, (s + d, th, ze, t), (s - d, th, ze, t), d)
        al_t = fd(4, (s, th + d, ze, t), (s, th - d, ze, t), d)
        al_z = fd(4, (s, th, ze + d, t), (s, th, ze - d, t), d)
        al_time = fd(4, (s, th, ze, t + dt), (s, th, ze, t - dt), dt)
        ref = np.array([Phi_s / fld.psi0, Phi_t, Phi_z, al_s / fld.psi0, al_t, al_z, al_time])
        got = np.array([o[1], o[2], o[3], o[5], o[6], o[7], o[8]])
        assert np.allclose(got, ref, rtol=2e-6, atol=1e-7 * np.abs(ref).max())


def test_pert_satisfies_ideal_mhd_constraint():
    """E_par = 0 (A14): b.grad(Phi) + B d(alpha)/dt = 0 with B.grad = B^2/(G + iota I) (iota d_theta + d_zeta),
    i.e. (iota Phi_theta + Phi_zeta) + (G + iota I) alpha_t = 0, evaluated from the oracle's outputs."""
    fld = _pert_field()
    F = oracle.OracleField(fld)
    rng = np.random.default_rng(5)
    for _ in range(10):
        s, th, ze, t = rng.uniform(0.05, 0.95), rng.uniform(-9, 9), rng.uniform(-9, 9), rng.uniform(0, 1e-3)
        o = F.eval_pert(s, th, ze, t)
        G, _, I, _, io, _ = F.eval_profiles(s)
        res = io * o[2] + o[3] + (G + io * I) * o[8]
        assert abs(res) < 1e-11 * (abs(o[2]) + abs(o[3]) + 1.0)


def test_zero_modes_gives_zero_perturbation():
    F = oracle.OracleField(W.make_field(0))
    assert np.all(F.eval_pert(0.3, 1.0, 2.0, 1e-5) == 0.0)
