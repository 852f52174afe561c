"""-m gpu: gc_orbit_diagnostics (classification, characteristic frequencies, J_par from uniform-time samples;
PAPER.md:50; reading A30) against oracle.orbit_diagnostics, series by series, through the C ABI."""
from __future__ import annotations

import numpy as np
import pytest

from gpu_common import make_case, record_info, to_dev

pytestmark = pytest.mark.gpu


def _compare(out, samples, send, j_first, dt, mass):
    import oracle
    keys = ["orbit_class", "reversals", "omega_theta", "omega_zeta", "omega_bounce", "j_par", "j_par_variation"]
    worst = 0.0
    for i in range(samples.shape[2]):
        sl = slice(j_first, int(send[i]))
        d = oracle.orbit_diagnostics(samples[1, sl, i], samples[2, sl, i], samples[3, sl, i], dt, mass)
        for q, key in enumerate(keys):
            a, b = out[q, i], d[key]
            if isinstance(b, float) and np.isnan(b):
                assert np.isnan(a), (i, key, a)
            elif q < 2:
                assert a == b, (i, key, a, b)                     # integer work: exact
            elif q == 6:
                assert abs(a - b) < 1e-12 + 1e-11 * abs(b), (i, key, a, b)    # (max - min) / mean: a cancelling difference
            else:
                err = abs(a - b) / max(abs(b), 1e-300) if b != 0.0 else abs(a)
                worst = max(worst, err)
                assert err < 1e-11, (i, key, a, b)
    return worst


def test_orbit_diagnostics_of_device_traces_match_the_oracle_definition():
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    fld, spec, P, OF, GF, mu = make_case(0, 300)
    T, nsamp = 1e-4, 1501
    dt = T / (nsamp - 1)
    r = GF.trace_sampled(spec, to_dev(P.s), to_dev(P.theta), to_dev(P.zeta), to_dev(P.vpar), to_dev(mu), 0.0, dt, nsamp,
                         t_max=T)
    out = G.orbit_diagnostics(r.samples, 0, r.sample_end, dt, spec.mass)
    torch.cuda.synchronize()
    S, send, O = r.samples.cpu().numpy(), r.sample_end.cpu().numpy(), out.cpu().numpy()
    worst = _compare(O, S, send, 0, dt, spec.mass)
    trapped = O[0] == 1.0
    assert 0.2 < trapped.mean() < 0.9 and (O[4][O[1] >= 3] > 0).all() and (O[5][O[1] >= 3] > 0).all()
    # no sample_end (all nsamp samples valid) and a later first sample
    full = send == nsamp
    out2 = G.orbit_diagnostics(r.samples, 100, None, dt, spec.mass).cpu().numpy()
    _compare(out2[:, full], S[:, :, full], np.full(int(full.sum()), nsamp), 100, dt, spec.mass)
    record_info("orbit_diagnostics", label="config 0, 300 particles, 1501 samples over 1e-4 s", max_rel=float(worst),
                trapped_fraction=float(trapped.mean()), median_bounce_omega=float(np.median(O[4][O[4] > 0])))


def test_orbit_diagnostics_edges_and_symplectic_samples():
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    # closed-form series laid out [4][nsamp][n]: pendulum, rotation, a particle with one valid sample, an empty one
    nsamp, n = 801, 4
    t = np.linspace(0.0, 2.0e-4, nsamp)
    S = np.zeros((4, nsamp, n))
    S[1, :, 0], S[2, :, 0], S[3, :, 0] = 0.7 * np.sin(2e5 * t + 0.3), 5e5 * t, 3e6 * np.cos(2e5 * t + 0.3)
    S[1, :, 1], S[2, :, 1], S[3, :, 1] = 2e5 * t + 1.0, -4e5 * t, 1e6
    S[3, :, 2:] = 1e6
    send = np.array([nsamp, nsamp, 1, 0], np.int32)
    out = G.orbit_diagnostics(to_dev(S), 0, to_dev(send, torch.int32), t[1], 6.64e-27).cpu().numpy()
    _compare(out[:, :2], S[:, :, :2], send[:2], 0, t[1], 6.64e-27)
    assert out[0, 0] == 1.0 and out[1, 0] == 13 and abs(out[4, 0] / 2e5 - 1.0) < 1e-6
    assert out[0, 1] == 0.0 and out[4, 1] == 0.0 and np.isnan(out[5, 1])
    assert np.isnan(out[0, 2]) and np.isnan(out[0, 3]) and np.isnan(out[2:, 2:]).all()
    for bad in (dict(sample_dt=0.0), dict(mass=-1.0)):
        kw = dict(sample_dt=1e-7, mass=1.0)
        kw.update(bad)
        with pytest.raises(G.GcError):
            G.orbit_diagnostics(to_dev(S), 0, None, kw["sample_dt"], kw["mass"])
    # samples of the symplectic integrator feed the same call
    fld, spec, P, OF, GF, mu = make_case(0, 64)
    s_n = np.arange(fld.ns) / (fld.ns - 1)
    chi = to_dev(fld.psi0 * (0.42 * s_n + 0.05 * s_n ** 2))
    r = GF.trace_symplectic(spec.mass, spec.charge, to_dev(P.s), to_dev(P.theta), to_dev(P.zeta), to_dev(P.vpar),
                            to_dev(mu), chi, 2e-8, 4000, sample_stride=10, nsamp=401)
    out = G.orbit_diagnostics(r.samples, 0, r.sample_end, 2e-7, spec.mass)
    torch.cuda.synchronize()
    _compare(out.cpu().numpy(), r.samples.cpu().numpy(), r.sample_end.cpu().numpy(), 0, 2e-7, spec.mass)
