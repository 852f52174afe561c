"""Pins for NEXT-2 of SURVEY.md section 8(f) in the oracle: B evaluated as a local tricubic interpolant of its own
node values on an (s, theta, zeta) grid ("CUDA kernels implement field interpolation", PAPER.md:80,111
"local tricubics"; reading A27 of DESIGN.md).  CPU only.

What fixes the arithmetic: the interpolation property at the nodes, an independent construction of the same
interpolant by successive numpy.polyfit through the 4 x 4 x 4 local node values (no weight formula retyped), central
finite differences of the interpolant for its three derivative outputs, periodicity in both angles, exactness on a
constant field, fourth-order convergence to the direct harmonic sum as the grid is refined, and along a trace the
conservation of energy (which holds only if the derivative outputs are the derivatives of the value output) and the
convergence of the traced orbit to the direct-sum orbit."""
import dataclasses
import math

import numpy as np
import pytest

import oracle
from paper_2605_16734_b200 import workloads as W

M, Q, VREF = W.ALPHA_MASS, W.ALPHA_CHARGE, W.V_ALPHA
TWO_PI = 2.0 * math.pi


def _field(ns=21):
    return W.make_equilibrium(3, 2, ns)


def _polyfit_interpolant(V, nfp, s, th, ze):
    """The tensor-product cubic through the 4 x 4 x 4 nodes around (s, th, ze), built by numpy.polyfit one direction
    after the other; returns value and the three first derivatives."""
    ngs, nth, nze = V.shape
    ds, dth, dze = 1.0 / (ngs - 1), TWO_PI / nth, TWO_PI / (nfp * nze)
    i0 = int(min(max(math.floor(s / ds) - 1, 0), ngs - 4))
    j0 = math.floor(th / dth) - 1
    k0 = math.floor(ze / dze) - 1
    sn = (i0 + np.arange(4)) * ds - s
    tn = (j0 + np.arange(4)) * dth - th
    zn = (k0 + np.arange(4)) * dze - ze
    blk = V[np.ix_(i0 + np.arange(4), (j0 + np.arange(4)) % nth, (k0 + np.arange(4)) % nze)]
    # along zeta: value and slope at ze for each (a, b)
    cz = np.polyfit(zn, blk.reshape(16, 4).T, 3)                     # [4 coef][16]
    v_z, d_z = cz[3].reshape(4, 4), cz[2].reshape(4, 4)
    # along theta
    ct_v = np.polyfit(tn, v_z.T, 3)                                  # columns = a
    ct_dz = np.polyfit(tn, d_z.T, 3)
    v_t, d_t, dz_t = ct_v[3], ct_v[2], ct_dz[3]
    # along s
    B = np.polyfit(sn, v_t, 3)
    return np.array([B[3], B[2], np.polyfit(sn, d_t, 3)[3], np.polyfit(sn, dz_t, 3)[3]])


def test_grid_nodes_hold_the_direct_sum_and_are_reproduced():
    fld = _field()
    F = oracle.OracleField(fld)
    F.set_grid(13, 12, 8)
    V = F.grid()
    assert V.shape == (13, 12, 8)
    rng = np.random.default_rng(0)
    for _ in range(20):
        i, j, k = rng.integers(0, 13), rng.integers(0, 12), rng.integers(0, 8)
        s, th, ze = i / 12.0, TWO_PI * j / 12, TWO_PI * k / (8 * fld.nfp)
        direct = F.eval_B_sum(s, th, ze)[0]
        assert V[i, j, k] == direct                                      # the table is the direct sum O2
        assert abs(F.eval_B(s, th, ze)[0] - direct) < 1e-13 * 5.7        # interpolation property
        # ... also one period further on, and at negative angles
        assert abs(F.eval_B(s, th - 3 * TWO_PI, ze + 5 * TWO_PI / fld.nfp)[0] - direct) < 1e-12 * 5.7


def test_interpolant_equals_successive_polyfit_through_the_local_nodes():
    fld = _field()
    F = oracle.OracleField(fld)
    F.set_grid(17, 16, 12)
    V = F.grid()
    rng = np.random.default_rng(1)
    pts = [(rng.uniform(0, 1), rng.uniform(-7, 7), rng.uniform(-7, 7)) for _ in range(30)]
    pts += [(0.01, 0.1, 0.1), (0.99, 6.2, 1.5), (0.5, -0.01, -0.01)]     # clamped radial stencils, wrap-around
    for s, th, ze in pts:
        got = F.eval_B(s, th, ze)
        ref = _polyfit_interpolant(V, fld.nfp, s, th, ze)
        assert np.allclose(got, ref, rtol=1e-9, atol=1e-9 * 5.7), (s, th, ze, got, ref)


def test_derivative_outputs_are_the_derivatives_of_the_interpolant():
    fld = _field()
    F = oracle.OracleField(fld)
    F.set_grid(17, 16, 12)
    rng = np.random.default_rng(2)
    for _ in range(10):
        # stay inside one cell in every direction so that the central difference sees one polynomial piece
        i, j, k = rng.integers(1, 15), rng.integers(0, 16), rng.integers(0, 12)
        s = (i + rng.uniform(0.3, 0.7)) / 16.0
        th = (j + rng.uniform(0.3, 0.7)) * TWO_PI / 16
        ze = (k + rng.uniform(0.3, 0.7)) * TWO_PI / (12 * fld.nfp)
        out = F.eval_B(s, th, ze)
        for c, (h, e) in enumerate(((1e-5, (1, 0, 0)), (1e-5, (0, 1, 0)), (1e-5, (0, 0, 1)))):
            up = F.eval_B(s + h * e[0], th + h * e[1], ze + h * e[2])[0]
            dn = F.eval_B(s - h * e[0], th - h * e[1], ze - h * e[2])[0]
            assert abs((up - dn) / (2 * h) - out[1 + c]) < 1e-7 * max(1.0, abs(out[1 + c]))


def test_periodic_in_both_angles_and_exact_on_a_constant_field():
    fld = _field()
    F = oracle.OracleField(fld)
    F.set_grid(9, 10, 6)
    a = F.eval_B(0.37, 1.234, 0.777)
    b = F.eval_B(0.37, 1.234 + TWO_PI, 0.777 - TWO_PI / fld.nfp)
    assert np.allclose(a, b, rtol=1e-12, atol=1e-12)
    flat = dataclasses.replace(fld, bmnc=np.where((fld.xm == 0) & (fld.xn == 0), 5.7, 0.0)[None, :] * np.ones((fld.ns, 1)))
    G = oracle.OracleField(flat)
    G.set_grid(9, 10, 6)
    out = G.eval_B(0.4321, 2.5, -1.1)
    assert abs(out[0] - 5.7) < 1e-14 and np.all(np.abs(out[1:]) < 1e-11)


def test_fourth_order_convergence_to_the_direct_sum():
    """Doubling every grid size divides the interpolation error of B by about 2^4 and that of the derivatives by
    about 2^3 (cubic pieces); the radial direction is exact here (same nodes, same stencil rule)."""
    fld = _field(ns=21)
    F = oracle.OracleField(fld)
    rng = np.random.default_rng(3)
    pts = [(rng.uniform(0.1, 0.9), rng.uniform(0, TWO_PI), rng.uniform(0, TWO_PI)) for _ in range(200)]
    direct = np.array([F.eval_B_sum(*p) for p in pts])
    errs = []
    for g in (16, 32, 64):
        F.set_grid(21, g, g)
        got = np.array([F.eval_B(*p) for p in pts])
        errs.append(np.sqrt(np.mean((got - direct) ** 2, axis=0)))
    F.set_grid(0, 0, 0)
    assert np.array_equal(np.array([F.eval_B(*p) for p in pts]), direct)     # back to the direct sum
    errs = np.array(errs)
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert 10.0 < r2[0] < 24.0 and r1[0] > 8.0, (errs, r1, r2)               # value: order 4
    assert r2[1] > 10.0                                                      # d/ds: angular error of a value-like term
    assert 5.5 < r2[2] < 12.0 and 5.5 < r2[3] < 12.0, (errs, r2)             # angular derivatives: order 3
    assert errs[2][0] < 2e-5 * 5.7


def _energy(F, mu, y):
    B = F.eval_B(y[0], y[1], y[2])[0]
    return 0.5 * M * y[3] ** 2 + mu * B


def test_trace_on_the_interpolant_conserves_energy_and_converges_to_the_direct_sum_orbit():
    """The interpolant is C0 with kinks of its derivatives at every node plane, so the adaptive integrator pays for
    each crossing (several times the attempts of the direct sum at the same tolerance) and the energy error carries
    a larger prefactor; it still falls with the tolerance, which it would not if B_s, B_theta, B_zeta were not the
    derivatives of the interpolated B (a 1 % error in one of them leaves a drift of 1e-4 whatever the tolerance)."""
    fld = _field(ns=21)
    P = W.make_particles(0, 6)
    F = oracle.OracleField(fld)
    mu = W.mu_from(P, np.array([F.eval_B_sum(a, b, c)[0] for a, b, c in zip(P.s, P.theta, P.zeta)]))
    drift = {}
    for rtol in (1e-9, 1e-12):
        spec = dataclasses.replace(W.make_spec(0), rtol=rtol, atol=rtol, t_max=2e-5)
        F.set_grid(21, 24, 24)
        r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
        assert np.all(r.status == 0)
        drift[rtol] = max(abs(_energy(F, mu[i], r.y[:, i]) - _energy(F, mu[i], [P.s[i], P.theta[i], P.zeta[i], P.vpar[i]]))
                          / _energy(F, mu[i], r.y[:, i]) for i in range(P.n))
    assert drift[1e-12] < 5e-8 and drift[1e-12] < drift[1e-9] / 50.0, drift
    spec = dataclasses.replace(W.make_spec(0), rtol=1e-10, atol=1e-10, t_max=2e-5)
    F.set_grid(0, 0, 0)
    ref = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
    diffs = []
    for g in (24, 48, 96):
        F.set_grid(21, g, g)
        r = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
        diffs.append(np.abs(r.y[:3] - ref.y[:3]).max())
    assert diffs[1] < diffs[0] / 6.0 and diffs[2] < diffs[1] / 6.0, diffs
    assert diffs[2] < 1e-4
