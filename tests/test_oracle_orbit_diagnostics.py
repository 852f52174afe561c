"""Pins for the oracle's orbit diagnostics (classification, characteristic frequencies, J_par from uniform-time samples;
PAPER.md:50 "characteristic orbit frequencies ... and orbit classification"; reading A30 of DESIGN.md section 12).
CPU only.  The diagnostics work on series, so they are pinned on series with a closed form, and on guiding-centre
orbits through an independent route (the bounce-section records of O8b, the closed-form passing orbit)."""
import math

import numpy as np

import oracle
from paper_2605_16734_b200 import workloads as W

M, Q, VREF = W.ALPHA_MASS, W.ALPHA_CHARGE, W.V_ALPHA


def test_closed_form_series_pendulum_and_rotation():
    # v = A cos(Om t + ph): reversals at Om t + ph = pi/2 + k pi, bounce frequency Om, J = m A^2 pi / Om per period
    A, Om, ph, m = 3.0e6, 2.0e5, 0.3, M
    errs = []
    for n in (401, 801, 1601):
        t = np.linspace(0.0, 2.0e-4, n)
        dt = t[1] - t[0]
        d = oracle.orbit_diagnostics(0.7 * np.sin(Om * t + ph), 5.0e5 * t, A * np.cos(Om * t + ph), dt, m)
        assert d["orbit_class"] == 1.0 and d["reversals"] == 13          # floor((Om T + ph - pi/2) / pi) + 1
        errs.append((abs(d["omega_bounce"] / Om - 1.0), abs(d["j_par"] / (m * A * A * math.pi / Om) - 1.0)))
        assert math.isclose(d["omega_zeta"], 5.0e5, rel_tol=1e-12)
        assert d["j_par_variation"] < 1e-3                                # every period is the same orbit
    # a cosine is a straight line to third order at its zeros: the interpolated crossing times are almost exact;
    # the trapezoid rule over a full period leaves only the two end pieces: J_par converges at third order in dt
    assert max(e[0] for e in errs) < 1e-6
    assert errs[0][1] < 1e-4 and 6.0 < errs[0][1] / errs[1][1] < 10.0 and 6.0 < errs[1][1] / errs[2][1] < 10.0
    # a rotation: no reversal, class 0, no bounce frequency, no J_par
    t = np.linspace(0.0, 1.0e-4, 101)
    d = oracle.orbit_diagnostics(2.0e5 * t + 1.0, -4.0e5 * t, np.full(101, 1.0e6), t[1], m)
    assert d["orbit_class"] == 0.0 and d["reversals"] == 0 and d["omega_bounce"] == 0.0 and math.isnan(d["j_par"])
    assert math.isclose(d["omega_theta"], 2.0e5, rel_tol=1e-12) and math.isclose(d["omega_zeta"], -4.0e5, rel_tol=1e-12)
    # brute force on a tiny hand-made series: reversals between samples (1, 2), (3, 4), (5, 6); one full period
    v = np.array([2.0, 1.0, -1.0, -2.0, 2.0, 1.0, -3.0])
    d = oracle.orbit_diagnostics(np.zeros(7), np.zeros(7), v, 1.0, 2.0)
    tau = [1.5, 3.5, 5.25]
    assert d["reversals"] == 3 and math.isclose(d["omega_bounce"], 2 * math.pi / (tau[2] - tau[0]))
    J = 2.0 * (0.5 * 1.0 * 0.5 + 0.5 * (1 + 4) + 0.5 * (4 + 4) + 0.5 * (4 + 1) + 0.5 * 1.0 * 0.25)
    assert math.isclose(d["j_par"], J) and d["j_par_variation"] == 0.0
    # fewer than two samples
    assert math.isnan(oracle.orbit_diagnostics([0.0], [0.0], [1.0], 1.0, 1.0)["orbit_class"])


def test_guiding_centre_orbits_passing_closed_form_and_trapped_against_the_bounce_section():
    # (i) B00-only field: zeta' = v B / G, theta' = iota zeta' exactly
    ns = 21
    s_n = np.arange(ns) / (ns - 1)
    fld = W.Field(ns=ns, nfp=4, xm=np.zeros(1, np.int32), xn=np.zeros(1, np.int32), bmnc=np.full((ns, 1), 5.7),
                  G=np.full(ns, 57.0), I=np.zeros(ns), iota=0.42 + 0.1 * s_n, psi0=W.PSI0)
    F = oracle.OracleField(fld)
    spec = W.make_spec(0)
    s0, v0 = np.array([0.3]), np.array([0.8 * VREF])
    mu = 0.5 * M * (VREF ** 2 - v0 ** 2) / 5.7
    r = F.trace_sampled(spec, s0, [0.5], [0.1], v0, mu, 0.0, 1e-7, 101, t_max=1e-5)
    d = oracle.orbit_diagnostics(r.samples[1, :, 0], r.samples[2, :, 0], r.samples[3, :, 0], 1e-7, M)
    assert d["orbit_class"] == 0.0
    assert math.isclose(d["omega_zeta"], v0[0] * 5.7 / 57.0, rel_tol=1e-9)
    assert math.isclose(d["omega_theta"], 0.45 * v0[0] * 5.7 / 57.0, rel_tol=1e-9)
    # (ii) config-0 field: trapped particles; the bounce frequency from the samples equals the one from the times of
    # the bounce-section records (O8b: v_par = 0 located on the continuous extension), an independent route
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    P = W.make_particles(0).head(64)
    mu = W.mu_from(P, F.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    T, nsamp = 1e-4, 2001
    r = F.trace_sampled(spec, P.s, P.theta, P.zeta, P.vpar, mu, 0.0, T / (nsamp - 1), nsamp, t_max=T)
    b = F.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=T, poincare_capacity=20000, section=1)
    checked = 0
    for i in range(P.n):
        if r.nsampled[i] < nsamp:
            continue
        d = oracle.orbit_diagnostics(r.samples[1, :, i], r.samples[2, :, i], r.samples[3, :, i], T / (nsamp - 1), M)
        tb = np.sort(b.poincare[b.poincare[:, 0] == i][:, 1])
        assert d["reversals"] == len(tb)                                 # same reversals found by both routes
        assert d["orbit_class"] == (1.0 if len(tb) else 0.0)
        if len(tb) >= 3:
            Pn = (len(tb) - 1) // 2
            ob = 2 * math.pi * Pn / (tb[2 * Pn] - tb[0])
            assert abs(d["omega_bounce"] / ob - 1.0) < 1e-4
            # J_par = m <v_par^2> T_b is below m v^2 T_b; it varies from bounce to bounce in this rippled field
            assert 0.0 < d["j_par"] < 2 * math.pi / ob * M * VREF ** 2 and d["j_par_variation"] >= 0.0
            checked += 1
    assert checked >= 5
