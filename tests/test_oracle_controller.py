"""Pins for the three controller branches of the oracle's trace loop that no other test states (O6, A9, A23) and
for the mode normalisation A16 of the input recipe.  CPU only.

The attempt sequence of a particle is reconstructed from the OUTSIDE: a run capped at max_steps = j stops after
attempt j (status 3) and returns the time reached, the counters and the next step proposal, so runs with
j = 1, 2, 3 ... give, attempt by attempt, the decision taken, the step size used and the step size proposed.  The
rules are then checked on that record; the error of an attempt is recomputed with the separately pinned
oracle_dp5_attempt / oracle_err_norm so that every test states the premise it relies on (err > 1, err < 0.59 ...).
"""
import math

import numpy as np

import oracle
from paper_2605_16734_b200 import workloads as W

M, Q, VREF = W.ALPHA_MASS, W.ALPHA_CHARGE, W.V_ALPHA


def _one_particle(k=3):
    fld = W.make_field(0)
    F = oracle.OracleField(fld)
    P = W.make_particles(0)
    s, th, ze, v = (np.array([a[k]]) for a in (P.s, P.theta, P.zeta, P.vpar))
    B = F.eval_B(s[0], th[0], ze[0])[0]
    mu = np.array([0.5 * M * (P.speed[k] ** 2 - v[0] ** 2) / B])
    return F, s, th, ze, v, mu


def _attempt_record(F, spec, s, th, ze, v, mu, n_attempts):
    """One entry per attempt 1 .. n_attempts: (accepted?, t after, n_acc, n_rej, n_forced, proposal after, y after)."""
    rec = []
    prev = (0, 0)
    for cap in range(1, n_attempts + 1):
        spec.max_steps = cap
        r = F.trace(spec, s, th, ze, v, mu)
        if r.status[0] != 3:                       # finished before the cap: the record ends here
            break
        acc, rej = int(r.n_acc[0]), int(r.n_rej[0])
        assert acc + rej == cap
        y = r.y[:, 0].copy()
        y[3] /= spec.v_ref
        rec.append((acc > prev[0], float(r.t[0]), acc, rej, int(r.n_forced[0]), float(r.h[0]), y))
        prev = (acc, rej)
    return rec


def _err_of_attempt(F, spec, t, y, mu, h):
    k1 = F.rhs(spec.mass, spec.charge, mu, spec.v_ref, t, y)
    y_new, k, delta = F.dp5_attempt(spec.mass, spec.charge, mu, spec.v_ref, t, y, k1, h)
    return oracle.err_norm(y, y_new, delta, spec.rtol, spec.atol), y_new


def test_attempt_at_h_min_is_forced_only_right_after_a_rejection():
    """O6 / A9 ("minimum step size control ... to prevent excessively small steps"): an attempt made with
    h == h_min is accepted whatever its error ONLY when the attempt before it was rejected.  Start with h0 = h_min
    far above the natural step: attempt 1 has err > 1 and no rejection before it, so it is REJECTED (the reading
    "forced whenever h == h_min" would accept it); the proposal is clamped back to h_min and attempt 2 is forced.
    After the forced accept the flag is clear again, so the pattern reject / forced accept repeats: with
    t_max = 4.5 h_min that is exactly 5 rejections, 5 accepted steps, all 5 forced."""
    F, s, th, ze, v, mu = _one_particle()
    spec = W.make_spec(0)
    spec.h_min = spec.h0 = 4e-7                                    # natural step ~3e-8 s
    spec.t_max = 4.5 * spec.h_min
    y0 = np.array([s[0], th[0], ze[0], v[0] / VREF])
    err1, _ = _err_of_attempt(F, spec, 0.0, y0, mu[0], spec.h_min)
    assert err1 > 1e3                                              # the premise: attempt 1 fails the error test
    rec = _attempt_record(F, spec, s, th, ze, v, mu, 9)
    assert [a for a, *_ in rec] == [False, True] * 4 + [False]     # attempts 1..9: reject, forced accept, ...
    assert rec[0][1] == 0.0 and rec[0][3] == 1 and rec[0][4] == 0  # attempt 1: rejected, not forced, t unchanged
    assert rec[0][5] == spec.h_min                                 # proposal clamped to h_min, not below
    assert rec[1][1] == spec.h_min and rec[1][4] == 1              # attempt 2: forced accept of a full h_min step
    spec.max_steps = 10 ** 9
    r = F.trace(spec, s, th, ze, v, mu)
    assert (r.status[0], r.n_acc[0], r.n_rej[0], r.n_forced[0]) == (0, 5, 5, 5) and r.t[0] == spec.t_max
    # the same start with h_min = 0 is an ordinary adaptive run: nothing is forced
    spec.h_min = 0.0
    r0 = F.trace(spec, s, th, ze, v, mu)
    assert r0.n_forced[0] == 0 and r0.n_rej[0] >= 1 and r0.n_acc[0] > 20


def test_no_growth_on_the_step_after_a_rejection():
    """O6: "if the previous attempt was a rejection, h_next = h min(scale, 1), else h scale".  On the piecewise-cubic
    radial interpolant steps that straddle a radial node are rejected now and then, and the retry often comes out
    with err < 0.59, i.e. with a controller factor 0.9 err^-0.2 > 1: the rule says the proposal after such an
    accepted retry EQUALS the step just taken (dropping the rule would let it grow by that factor).  Accepted
    attempts with no rejection before them follow h_next = h scale exactly."""
    F, s, th, ze, v, mu = _one_particle()
    spec = W.make_spec(0)
    spec.t_max = 1e-3
    rec = _attempt_record(F, spec, s, th, ze, v, mu, 130)
    assert len(rec) == 130
    held = grown = 0
    for j in range(1, len(rec)):
        if not rec[j][0]:
            continue
        t_b, y_b, h_used = rec[j - 1][1], rec[j - 1][6], rec[j - 1][5]
        err, _ = _err_of_attempt(F, spec, t_b, y_b, mu[0], h_used)
        assert err <= 1.0 and rec[j][1] == t_b + h_used             # the accepted attempt used the last proposal
        sc = oracle.scale_accept(err)
        if not rec[j - 1][0]:                                       # right after a rejection
            assert rec[j][5] <= h_used
            if sc > 1.0:
                assert rec[j][5] == h_used                          # held, although the factor is above one
                held += sc > 1.01
            else:
                assert math.isclose(rec[j][5], h_used * sc, rel_tol=1e-7)
        else:                                                       # (err is recomputed from a state whose v_par went
            assert math.isclose(rec[j][5], h_used * sc, rel_tol=1e-7)   # through m/s and back: equal to ~1e-10 only)
            grown += sc > 1.0
    assert held >= 5 and grown >= 20                                # premises: both cases occur in this record
    # a rejected attempt shrinks the proposal by max(0.9 err^-0.2, 0.2) and leaves t and y alone
    n_rej = 0
    for j in range(1, len(rec)):
        if rec[j][0]:
            continue
        t_b, y_b, h_used = rec[j - 1][1], rec[j - 1][6], rec[j - 1][5]
        err, _ = _err_of_attempt(F, spec, t_b, y_b, mu[0], h_used)
        assert err > 1.0 and rec[j][1] == t_b and np.array_equal(rec[j][6], y_b)
        assert math.isclose(rec[j][5], h_used * oracle.scale_reject(err), rel_tol=1e-7) and 0.2 * h_used <= rec[j][5] < h_used
        n_rej += 1
    assert n_rej >= 10


def test_clipped_last_step_hands_on_the_unclipped_proposal():
    """O6: "the step that would pass t_max is clipped to land on it; the unclipped h_next is
    kept for h_inout", so that a horizon cut into segments continues with the step size the controller had reached,
    not with one derived from the short clipped step.  Built by hand: take the attempt record up to an accepted
    attempt k (no rejection before it), whose proposal is h_k = h_used scale_accept(err_k); put t_max 0.05 h_k behind
    t_k, so attempt k + 1 is clipped to 0.05 h_k.  The call must end on t_max and return h_k -- not
    0.05 h_k scale_accept(err of the clipped step), at most half of h_k whatever the growth cap, the value the reading "every accepted step updates h" gives
    (mutation `if (!clipped) h = h_next` -> `h = h_next` of trace_impl).  The next segment then starts with a full
    step h_k."""
    F, s, th, ze, v, mu = _one_particle()
    spec = W.make_spec(0)
    spec.t_max = 1e-3
    rec = _attempt_record(F, spec, s, th, ze, v, mu, 40)
    k = next(j for j in range(20, 40) if rec[j][0] and rec[j - 1][0])      # accepted, and so was the one before it
    t_b, y_b, h_used = rec[k - 1][1], rec[k - 1][6], rec[k - 1][5]
    err_k, _ = _err_of_attempt(F, spec, t_b, y_b, mu[0], h_used)
    h_k = h_used * oracle.scale_accept(err_k)                               # the proposal after attempt k, by hand
    t_k, y_k = rec[k][1], rec[k][6]
    assert t_k == t_b + h_used and math.isclose(rec[k][5], h_k, rel_tol=1e-7)
    spec.max_steps = 10 ** 9
    spec.t_max = t_k + 0.05 * h_k
    a = F.trace(spec, s, th, ze, v, mu, traj_capacity=64)
    assert a.status[0] == 0 and a.t[0] == spec.t_max and a.n_acc[0] + a.n_rej[0] == k + 2   # attempts are 0-based in rec
    h_clip = spec.t_max - t_k
    err_c, _ = _err_of_attempt(F, spec, t_k, y_k, mu[0], h_clip)
    h_wrong = h_clip * oracle.scale_accept(err_c)                           # what the other reading would hand on
    assert err_c <= 1.0 and h_wrong < 0.6 * h_k    # premise: the two readings differ
    assert math.isclose(a.h[0], h_k, rel_tol=1e-7)
    assert a.h[0] == rec[k][5]                                              # exactly the proposal before the clip
    # the second segment takes its first step with that h: the accepted step sequence of the two-segment run
    # continues t_k + 0.05 h_k -> + h_k (err of that attempt, recomputed here, is below one)
    T2 = spec.t_max + 5.0 * h_k
    y_a = np.array([a.y[0, 0], a.y[1, 0], a.y[2, 0], a.y[3, 0] / VREF])
    err_n, _ = _err_of_attempt(F, spec, a.t[0], y_a, mu[0], a.h[0])
    assert err_n <= 1.0
    b = F.trace(spec, a.y[0], a.y[1], a.y[2], a.y[3], mu, h_in=a.h, t0=a.t[0], t_max=T2, traj_capacity=64)
    assert b.traj[0, 0, 0] == a.t[0] + h_k
    # and the whole two-segment run stays on the single call's error level
    full = F.trace(spec, s, th, ze, v, mu, t_max=T2)
    assert np.abs(b.y[:3, 0] - full.y[:3, 0]).max() < 1e-9 and abs(b.y[3, 0] - full.y[3, 0]) < 1e-9 * VREF


def test_step_underflow_ends_the_particle_with_status_4():
    """A23: with h_min = 0 a step so small that t + h == t in floating point can never advance the particle; it ends
    with status 4 (non-finite / stalled) instead of looping for ever: zero attempts, state untouched."""
    F, s, th, ze, v, mu = _one_particle()
    spec = W.make_spec(0)
    spec.h_min, spec.h0 = 0.0, 1e-12
    spec.max_steps = 1000                                          # (an implementation without the rule ends here, status 3)
    r = F.trace(spec, s, th, ze, v, mu, t0=1e8, t_max=2e8)         # ulp(1e8) = 1.5e-8 >> h0
    assert 1e8 + spec.h0 == 1e8
    assert r.status[0] == 4 and r.n_acc[0] == 0 and r.n_rej[0] == 0 and r.t[0] == 1e8
    assert r.y[0, 0] == s[0] and r.y[3, 0] == v[0]
    # with a minimum step that does advance t the same start is an ordinary run
    spec.h_min = 1e-7
    spec.max_steps = 50
    r2 = F.trace(spec, s, th, ze, v, mu, t0=1e8, t_max=2e8)
    assert r2.status[0] == 3 and r2.t[0] > 1e8 and r2.n_acc[0] > 0


def _realised_dB_over_B(fld, ks):
    """max over the radial nodes of sqrt(sum_k (m_k alpha_hat_k(s) / (a sqrt s))^2) for the harmonics `ks` of the
    field's mode table, with alpha_hat_k(s) read off the ORACLE's perturbation evaluation (O3) of a field that
    holds harmonic k alone, at an angle where sin(phase) = 1."""
    s_nodes = np.arange(1, fld.ns) / (fld.ns - 1)                  # skip s = 0 (the measure divides by sqrt s)
    tot = np.zeros_like(s_nodes)
    for k in ks:
        one = W.Field(ns=fld.ns, nfp=fld.nfp, xm=fld.xm, xn=fld.xn, bmnc=fld.bmnc, G=fld.G, I=fld.I, iota=fld.iota,
                      psi0=fld.psi0, mode_m=fld.mode_m[k:k + 1], mode_n=fld.mode_n[k:k + 1],
                      mode_omega=fld.mode_omega[k:k + 1], mode_phase=np.zeros(1),
                      phihat=np.ascontiguousarray(fld.phihat[:, k:k + 1]))
        F = oracle.OracleField(one)
        m = int(fld.mode_m[k])
        th = (math.pi / 2) / m                                     # m theta = pi/2, zeta = 0, t = 0: sin = 1, cos = 0
        ah = np.array([F.eval_pert(s, th, 0.0, 0.0)[4] for s in s_nodes])
        tot += (m * ah / (W.A_MINOR * np.sqrt(s_nodes))) ** 2
    return math.sqrt(tot.max())


def test_mode_amplitudes_realise_the_stated_dB_over_B():
    """A16 (BASELINE.json configs[2] "normalised so that deltaB/B=1e-4", configs[4] "deltaB/B=5e-5 each"): the
    amplitudes the input recipe produces, pushed through the oracle's own alpha (ideal-MHD relation O3), give the
    stated radial-field measure -- so an error in the recipe's normalisation cannot hide on both sides."""
    f2 = W.make_field(2)
    assert abs(_realised_dB_over_B(f2, range(f2.nk)) / 1e-4 - 1.0) < 1e-9
    f4 = W.make_field(4)
    for k in range(f4.nk):
        assert abs(_realised_dB_over_B(f4, [k]) / 5e-5 - 1.0) < 1e-9, k
