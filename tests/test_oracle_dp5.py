"""Pins for the oracle's Dormand-Prince 5(4) step, dense output and controller (O5, O6, O8).  CPU only."""
import math

import numpy as np
import pytest
from scipy.integrate import RK45
from scipy.integrate._ivp.rk import rk_step

import oracle


def _poly_rhs(k):
    return lambda t, y: np.array([t ** k, 2.0 * t ** k, -t ** k, 0.0])


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_fifth_order_solution_exact_on_polynomials(k):
    t0, h = 0.7, 0.45
    y0 = np.array([1.0, -2.0, 0.5, 3.0])
    y_new, ks, delta = oracle.dp5_attempt_fn(_poly_rhs(k), t0, y0, h)
    inc = ((t0 + h) ** (k + 1) - t0 ** (k + 1)) / (k + 1)
    assert np.allclose(y_new, y0 + np.array([inc, 2 * inc, -inc, 0.0]), rtol=1e-14, atol=1e-14)
    if k <= 3:                       # the embedded 4th-order solution is exact too: delta vanishes
        assert np.all(np.abs(delta) < 1e-15)
    else:
        assert abs(delta[0]) > 1e-8
    # FSAL: the seventh stage is f(t+h, y_new)
    assert np.allclose(ks[6], _poly_rhs(k)(t0 + h, y_new), rtol=1e-15, atol=0)


def _toy(t, y):
    return np.array([y[1], -math.sin(y[0]) + 0.1 * math.cos(t), y[3] * y[2] * 0.3, -y[2] + t])


def test_one_step_equals_scipy_rk45_step():
    """scipy's RK45 uses the same Dormand-Prince tableau: a library routine on the same step."""
    t0, h = 0.3, 0.17
    y0 = np.array([0.4, -0.2, 1.1, 0.9])
    y_new, ks, delta = oracle.dp5_attempt_fn(_toy, t0, y0, h)
    K = np.empty((7, 4))
    y_sp, f_sp = rk_step(_toy, t0, y0, _toy(t0, y0), h, RK45.A, RK45.B, RK45.C, K)
    assert np.allclose(y_new, y_sp, rtol=1e-14, atol=1e-15)
    assert np.allclose(ks, K, rtol=1e-13, atol=1e-15)
    err_sp = K.T @ RK45.E * h          # scipy: (5th - 4th) with its own sign convention
    assert np.allclose(np.abs(delta), np.abs(err_sp), rtol=1e-9, atol=1e-17)
    assert np.allclose(delta, err_sp, rtol=1e-9, atol=1e-17) or np.allclose(delta, -err_sp, rtol=1e-9, atol=1e-17)


def test_global_convergence_order_is_five():
    def solve(nsteps):
        t, y = 0.0, np.array([0.4, -0.2, 1.1, 0.9])
        h = 1.0 / nsteps
        for _ in range(nsteps):
            y, _, _ = oracle.dp5_attempt_fn(_toy, t, y, h)
            t += h
        return y
    ref = solve(256)
    e1 = np.abs(solve(8) - ref).max()
    e2 = np.abs(solve(16) - ref).max()
    assert 4.5 < math.log2(e1 / e2) < 5.8


def test_embedded_error_is_fifth_order_local():
    y0 = np.array([0.4, -0.2, 1.1, 0.9])
    d1 = np.abs(oracle.dp5_attempt_fn(_toy, 0.3, y0, 0.2)[2]).max()
    d2 = np.abs(oracle.dp5_attempt_fn(_toy, 0.3, y0, 0.1)[2]).max()
    assert 4.5 < math.log2(d1 / d2) < 5.5


@pytest.mark.parametrize("k", [0, 1, 2, 3])
def test_dense_output_exact_on_cubic_rhs(k):
    t0, h = 0.2, 0.6
    y0 = np.array([0.0, 1.0, 2.0, 3.0])
    y_new, ks, _ = oracle.dp5_attempt_fn(_poly_rhs(k), t0, y0, h)
    for tau in (0.0, 1.0 / 3.0, 0.5, 0.9, 1.0):
        inc = ((t0 + tau * h) ** (k + 1) - t0 ** (k + 1)) / (k + 1)
        y_tau = oracle.dp5_dense(y0, y_new, ks, h, tau)
        assert np.allclose(y_tau, y0 + np.array([inc, 2 * inc, -inc, 0.0]), rtol=1e-13, atol=1e-14)


def test_dense_output_endpoints_and_fourth_order_accuracy():
    t0 = 0.3
    y0 = np.array([0.4, -0.2, 1.1, 0.9])
    errs = []
    for h in (0.2, 0.1):
        y_new, ks, _ = oracle.dp5_attempt_fn(_toy, t0, y0, h)
        assert np.allclose(oracle.dp5_dense(y0, y_new, ks, h, 0.0), y0, atol=1e-15)
        assert np.allclose(oracle.dp5_dense(y0, y_new, ks, h, 1.0), y_new, rtol=1e-15, atol=1e-15)
        # reference at the midpoint by many small steps
        t, y = t0, y0.copy()
        for _ in range(64):
            y, _, _ = oracle.dp5_attempt_fn(_toy, t, y, h / 128)
            t += h / 128
        errs.append(np.abs(oracle.dp5_dense(y0, y_new, ks, h, 0.5) - y).max())
    assert 4.3 < math.log2(errs[0] / errs[1]) < 6.2       # local error of a 4th-order interpolant ~ h^5


def test_dense_output_equals_scipy_dense_output():
    """scipy's RK45 dense output is a quartic built from the same seven stages; both interpolants are the
    Dormand-Prince/Shampine continuous extension, so they must agree to rounding."""
    t0, h = 0.3, 0.17
    y0 = np.array([0.4, -0.2, 1.1, 0.9])
    y_new, ks, _ = oracle.dp5_attempt_fn(_toy, t0, y0, h)
    Q = ks.T @ RK45.P                                   # [4 comps][4 powers]
    for tau in (0.1, 0.37, 0.5, 0.82):
        p = np.array([tau, tau ** 2, tau ** 3, tau ** 4])
        y_sp = y0 + h * (Q @ p)
        assert np.allclose(oracle.dp5_dense(y0, y_new, ks, h, tau), y_sp, rtol=1e-12, atol=1e-14)


def test_error_norm_hand_values():
    y = np.array([1.0, -2.0, 0.0, 4.0])
    yn = np.array([1.5, -1.0, 0.0, -5.0])
    d = np.array([1e-9, 2e-9, 3e-10, -4e-9])
    rtol, atol = 1e-8, 1e-10
    sk = atol + rtol * np.array([1.5, 2.0, 0.0, 5.0])
    exp = math.sqrt(np.mean((d / sk) ** 2))
    assert abs(oracle.err_norm(y, yn, d, rtol, atol) - exp) < 1e-12 * exp


def test_controller_factors_hand_values():
    """O6: S = 0.9, exponent 0.2, minscale 0.2, maxscale 10."""
    assert oracle.scale_accept(0.0) == 10.0
    assert abs(oracle.scale_accept(1.0) - 0.9) < 1e-15
    assert abs(oracle.scale_accept(1.0 / 32.0) - 1.8) < 1e-14          # 0.9 * 32^0.2 = 1.8
    assert abs(oracle.scale_accept(1e-10) - 10.0) < 1e-15              # 0.9 * 100 = 90 -> clamp 10
    assert abs(oracle.scale_accept(32.0 ** 5) - 0.2) < 1e-15           # forced accepts with huge err clamp low
    assert abs(oracle.scale_reject(32.0) - 0.45) < 1e-14               # 0.9 / 2
    assert abs(oracle.scale_reject(1e12) - 0.2) < 1e-15
    assert oracle.scale_reject(float("nan")) == 0.2
    assert oracle.scale_reject(float("inf")) == 0.2
    # never grows after a rejection, never shrinks below minscale
    for e in np.logspace(0.0001, 8, 30):
        assert 0.2 <= oracle.scale_reject(float(e)) < 0.9 + 1e-12
