"""Pins for the second reading of NEXT-2 in the oracle: B as the C1 tricubic HERMITE interpolant of its node values and
node derivatives ("local tricubics"; reading A31 of DESIGN.md).  CPU only.

What fixes the arithmetic: finite differences of the direct sum (the node data), the interpolation property for value
and gradient at the nodes, the same interpolant rebuilt by successive 1-D scipy.interpolate.CubicHermiteSpline passes
(no basis formula retyped), continuity of value and gradient across cell faces in all three directions (which the
Lagrange reading A27 does not have), periodicity, fourth-order convergence to the direct sum, and along a trace the
conservation of energy and a controller that rejects far fewer attempts than on the C0 interpolant."""
import math

import numpy as np
from scipy.interpolate import CubicHermiteSpline

import oracle
from paper_2605_16734_b200 import workloads as W

TWO_PI = 2.0 * math.pi


def _field(ns=21):
    return W.make_equilibrium(3, 2, ns)


def test_mixed_derivatives_of_the_direct_sum_against_finite_differences():
    fld = _field()
    fld.bmns = 0.3 * fld.bmnc * (fld.xm[None, :] > 0)           # also the sin table
    F = oracle.OracleField(fld)
    s, th, ze = 0.437, 1.1, -0.6                                # inside a radial cell: the sum is smooth there
    d = F.eval_B_mixed(s, th, ze)
    base = F.eval_B_sum(s, th, ze)
    assert np.allclose(d[:4], base, rtol=1e-14, atol=0)
    e = 1e-5
    f_th = lambda ss, tt, zz: F.eval_B_sum(ss, tt, zz)[2]
    f_s = lambda ss, tt, zz: F.eval_B_sum(ss, tt, zz)[1]
    fd_sth = (f_th(s + e, th, ze) - f_th(s - e, th, ze)) / (2 * e)
    fd_sze = (F.eval_B_sum(s + e, th, ze)[3] - F.eval_B_sum(s - e, th, ze)[3]) / (2 * e)
    fd_thze = (f_th(s, th, ze + e) - f_th(s, th, ze - e)) / (2 * e)
    fd_all = (f_s(s, th + e, ze + e) - f_s(s, th + e, ze - e) - f_s(s, th - e, ze + e) + f_s(s, th - e, ze - e)) / (4 * e * e)
    for got, fd in zip(d[4:], (fd_sth, fd_sze, fd_thze, fd_all)):
        assert abs(got - fd) < 2e-6 * max(1.0, abs(fd)), (got, fd)
        assert abs(got) > 1e-3                                  # every one is really there


def test_nodes_reproduce_value_and_gradient_and_the_interpolant_is_C1():
    fld = _field()
    F = oracle.OracleField(fld)
    ngs, nth, nze = 11, 10, 7
    F.set_grid_hermite(ngs, nth, nze)
    D = F.grid8()
    assert D.shape == (ngs, nth, nze, 8)
    rng = np.random.default_rng(1)
    for _ in range(20):
        i, j, k = rng.integers(1, ngs - 1), rng.integers(0, nth), rng.integers(0, nze)
        s, th, ze = i / (ngs - 1.0), TWO_PI * j / nth, TWO_PI * k / (nze * fld.nfp)
        got = F.eval_B(s, th, ze)
        assert np.allclose(got, D[i, j, k, :4], rtol=1e-12, atol=1e-12)
    # continuity of value and gradient across faces in each direction (a jump would be of the size of the
    # interpolation error, ~1e-3 here); the Lagrange reading has such jumps in the gradient
    F2 = oracle.OracleField(fld)
    F2.set_grid(ngs, nth, nze)
    e = 1e-9
    faces = [((3 / (ngs - 1.0), 0.77, 0.31), 0), ((0.377, TWO_PI * 4 / nth, 0.31), 1),
             ((0.377, 0.77, TWO_PI * 3 / (nze * fld.nfp)), 2)]
    for pt, ax in faces:
        lo, hi = list(pt), list(pt)
        lo[ax] -= e
        hi[ax] += e
        jump_h = np.abs(F.eval_B(*hi) - F.eval_B(*lo))
        jump_l = np.abs(F2.eval_B(*hi) - F2.eval_B(*lo))
        assert jump_h.max() < 1e-5, (ax, jump_h)                # smooth change over 2e-9 only
        assert jump_l[1:].max() > 1e-4, (ax, jump_l)            # C0: the gradient jumps
    # periodicity in both angles, and the clamped radial cell extrapolates smoothly beyond s = 1
    a = F.eval_B(0.41, 0.9, 0.2)
    assert np.allclose(a, F.eval_B(0.41, 0.9 + 3 * TWO_PI, 0.2 - 5 * TWO_PI / fld.nfp), rtol=1e-11, atol=1e-11)
    assert np.allclose(F.eval_B(1.0 + 1e-9, 0.9, 0.2), F.eval_B(1.0 - 1e-9, 0.9, 0.2), atol=1e-6)


def _scipy_hermite(D, nfp, s, th, ze):
    """The tensor-product Hermite interpolant rebuilt with scipy's 1-D CubicHermiteSpline, one direction after the
    other: along zeta interpolate {f, f_s, f_th, f_s_th} with their zeta-derivatives, then along theta, then along s."""
    ngs, nth, nze, _ = D.shape
    ds, dth, dze = 1.0 / (ngs - 1), TWO_PI / nth, TWO_PI / (nfp * nze)
    i = int(min(max(math.floor(s / ds), 0), ngs - 2))
    j, k = math.floor(th / dth), math.floor(ze / dze)
    zn = np.array([k, k + 1]) * dze
    tn = np.array([j, j + 1]) * dth
    sn = np.array([i, i + 1]) * ds
    blk = D[np.ix_([i, i + 1], [j % nth, (j + 1) % nth], [k % nze, (k + 1) % nze])]      # [2][2][2][8]
    pair = {0: 3, 1: 5, 2: 6, 4: 7}                          # quantity -> its zeta-derivative
    Z, Zd = {}, {}
    for q, qz in pair.items():
        Z[q] = np.empty((2, 2)); Zd[q] = np.empty((2, 2))
        for a in range(2):
            for b in range(2):
                sp = CubicHermiteSpline(zn, blk[a, b, :, q], blk[a, b, :, qz])
                Z[q][a, b], Zd[q][a, b] = sp(ze), sp(ze, 1)
    # along theta: f with f_th, f_s with f_s_th; the zeta-derivatives likewise
    def along_theta(val, slope):
        out, dout = np.empty(2), np.empty(2)
        for a in range(2):
            sp = CubicHermiteSpline(tn, val[a], slope[a])
            out[a], dout[a] = sp(th), sp(th, 1)
        return out, dout
    f_, fth_ = along_theta(Z[0], Z[2])
    fs_, _ = along_theta(Z[1], Z[4])
    fze_, _ = along_theta(Zd[0], Zd[2])
    fsze_, _ = along_theta(Zd[1], Zd[4])
    fsth_ = along_theta(Z[1], Z[4])[1]
    B = CubicHermiteSpline(sn, f_, fs_)
    Bt = CubicHermiteSpline(sn, fth_, fsth_)
    Bz = CubicHermiteSpline(sn, fze_, fsze_)
    return np.array([B(s), B(s, 1), Bt(s), Bz(s)])


def test_interpolant_equals_successive_scipy_hermite_splines():
    fld = _field()
    F = oracle.OracleField(fld)
    F.set_grid_hermite(9, 8, 6)
    D = F.grid8()
    rng = np.random.default_rng(3)
    for _ in range(25):
        s, th, ze = rng.uniform(0.02, 0.98), rng.uniform(-4.0, 9.0), rng.uniform(-3.0, 3.0)
        got = F.eval_B(s, th, ze)
        ref = _scipy_hermite(D, fld.nfp, s, th, ze)
        assert np.allclose(got, ref, rtol=1e-10, atol=1e-10), (s, th, ze, got, ref)


def test_fourth_order_convergence_to_the_direct_sum():
    fld = W.make_equilibrium(3, 2, 81)
    s = np.arange(fld.ns) / (fld.ns - 1)
    fld.bmnc = np.ascontiguousarray(fld.bmnc[-1][None, :] * (0.3 + 0.5 * s + 0.4 * s ** 2 - 0.2 * s ** 3)[:, None])
    F = oracle.OracleField(fld)                              # amplitudes cubic in s: the direct sum is smooth in s
    rng = np.random.default_rng(5)
    pts = np.column_stack([rng.uniform(0.1, 0.9, 40), rng.uniform(0, TWO_PI, 40), rng.uniform(0, TWO_PI / fld.nfp, 40)])
    ref = np.array([F.eval_B_sum(*p) for p in pts])
    err = []
    for n in (8, 16, 32):
        F.set_grid_hermite(n + 1, 2 * n, 2 * n)
        err.append(np.abs(np.array([F.eval_B(*p) for p in pts]) - ref).max(axis=0))
    err = np.array(err)
    assert (err[0, 0] / err[1, 0] > 10.0) and (err[1, 0] / err[2, 0] > 10.0)        # value: ~16 per halving
    for c in (1, 2, 3):                                                            # gradient: third order, ~8
        assert err[0, c] / err[1, c] > 5.0 and err[1, c] / err[2, c] > 5.0
    assert err[2, 0] < 1e-5


def test_trace_conserves_energy_and_rejects_fewer_attempts_than_on_the_C0_interpolant():
    fld = W.make_field(0)
    P = W.make_particles(0).head(24)
    spec = W.make_spec(0)
    M = W.ALPHA_MASS
    res = {}
    for kind in ("hermite", "lagrange"):
        F = oracle.OracleField(fld)
        (F.set_grid_hermite if kind == "hermite" else F.set_grid)(51, 64, 64)
        B0 = F.eval_B_many(P.s, P.theta, P.zeta)[:, 0]
        mu = W.mu_from(P, B0)
        r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=2e-5)
        B1 = F.eval_B_many(r.y[0], r.y[1], r.y[2])[:, 0]
        E0 = 0.5 * M * P.vpar ** 2 + mu * B0
        E1 = 0.5 * M * r.y[3] ** 2 + mu * B1
        res[kind] = (np.abs(E1 / E0 - 1.0).max(), r.n_acc.sum(), r.n_rej.sum())
    # energy: the derivative outputs are the derivatives of the value output, so H is conserved by the exact flow; what
    # is left is the integrator's error at the faces, where the second (Hermite) or first (Lagrange) derivatives jump
    assert res["hermite"][0] < 2e-5 and res["hermite"][0] < res["lagrange"][0], res
    # smoother field: far fewer rejections and attempts for the same 2e-5 s at the same tolerance
    assert res["hermite"][2] < 0.25 * res["lagrange"][2], res
    assert res["hermite"][1] + res["hermite"][2] < 0.35 * (res["lagrange"][1] + res["lagrange"][2]), res
