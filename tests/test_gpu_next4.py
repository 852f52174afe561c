"""-m gpu: NEXT-4 of SURVEY.md section 8(f) on the device against the oracle: sin (non-stellarator-symmetric) harmonics
of B and the covariant radial component K (field model of PAPER.md:44 without the two simplifications of reading A4).
Through the C ABI; the oracle side is pinned in tests/test_oracle_next4.py.

The device evaluates the sin series with the cos sweep and (c_m, s_m) rotated by a quarter period, and inverts the
antisymmetric 4 x 4 Euler-Lagrange system in closed form through its Pfaffian; the oracle sums sin terms one by one and
solves the system by Gaussian elimination: the two share no formulation."""
from __future__ import annotations

import numpy as np
import pytest

from gpu_common import assert_trace_parity, gpu_trace, oracle_conditioning, to_dev

pytestmark = pytest.mark.gpu


def _asym_field(with_K=True, with_modes=True, M=11, N=13, ns=61, seed=7):
    """I != 0, G' != 0, shuffled harmonics with one duplicated (m, n) pair (also with n < 0 and m = 0), seeded sin
    harmonics of a few per cent of B00, K of the size I / a^2, two modes."""
    from paper_2605_16734_b200 import workloads as W
    rng = np.random.default_rng(seed)
    xm, xn = W.harmonic_list(M, N)
    # the generator omits (m = 0, n < 0); a sin table is not symmetric under n -> -n there, so add a few of them
    xm, xn = np.append(xm, [0, 0, 0]), np.append(xn, [-1, -4, -N])
    s_n = np.arange(ns) / (ns - 1)
    damp = np.exp(-(xm + np.abs(xn)) / 3.0)
    shape = s_n[:, None] ** (np.maximum(xm, 1)[None, :] / 2.0)
    bmnc = 0.04 * 5.0 * rng.standard_normal(xm.size)[None, :] * damp[None, :] * (s_n[:, None] ** (xm[None, :] / 2.0))
    bmnc[:, (xm == 0) & (xn == 0)] = (5.0 + 0.3 * s_n)[:, None]
    bmnc[:, (xm == 0) & (xn < 0)] *= 0.3
    bmns = 0.05 * 5.0 * rng.standard_normal(xm.size)[None, :] * damp[None, :] * shape
    kmnc = 0.7 * rng.standard_normal(xm.size)[None, :] * damp[None, :] * shape
    kmns = 1.5 * rng.standard_normal(xm.size)[None, :] * damp[None, :] * shape * (1.0 + s_n[:, None])
    perm = rng.permutation(xm.size)
    xm, xn = xm[perm], xn[perm]
    bmnc, bmns, kmnc, kmns = bmnc[:, perm], bmns[:, perm], kmnc[:, perm], kmns[:, perm]
    dup = int(np.nonzero((xm == 3) & (xn == -2))[0][0])
    xm, xn = np.append(xm, xm[dup]), np.append(xn, xn[dup])
    ext = lambda a: np.ascontiguousarray(np.concatenate([a, 0.5 * a[:, dup:dup + 1]], axis=1))
    env = np.exp(-(s_n - 0.45) ** 2 / (2 * 0.08 ** 2))
    kw = {}
    if with_modes:
        kw = dict(mode_m=np.array([4, 7], np.int32), mode_n=np.array([-3, 5], np.int32),
                  mode_omega=2 * np.pi * np.array([90e3, -210e3]), mode_phase=np.array([0.4, 2.0]),
                  phihat=np.stack([3e3 * env, -2e3 * env], axis=1))
    return W.Field(ns=ns, nfp=3, xm=xm.astype(np.int32), xn=xn.astype(np.int32), bmnc=ext(bmnc),
                   G=48.0 + 2.0 * s_n - 0.7 * s_n ** 2, I=1.5 * s_n + 0.4 * s_n ** 2,
                   iota=0.38 + 0.2 * s_n - 0.05 * s_n ** 3, psi0=6.5, bmns=ext(bmns),
                   kmnc=ext(kmnc) if with_K else None, kmns=ext(kmns) if with_K else None, **kw)


def test_series_with_sin_tables_and_K_match_the_oracle():
    import torch
    import oracle
    from paper_2605_16734_b200 import gcorbit as G
    fld = _asym_field()
    OF, GF = oracle.OracleField(fld), G.Field(fld)
    rng = np.random.default_rng(1)
    n = 257
    s, th, ze = rng.uniform(-0.02, 1.02, n), rng.uniform(-40, 40, n), rng.uniform(-40, 40, n)
    B, dB = GF.field_eval(to_dev(s), to_dev(th), to_dev(ze))
    K, dK = GF.kcov_eval(to_dev(s), to_dev(th), to_dev(ze))
    torch.cuda.synchronize()
    got_B = np.vstack([B.cpu().numpy()[None], dB.cpu().numpy()])
    got_K = np.vstack([K.cpu().numpy()[None], dK.cpu().numpy()])
    ref_B = np.array([OF.eval_B(*p) for p in zip(s, th, ze)]).T
    ref_K = np.array([OF.eval_K(*p) for p in zip(s, th, ze)]).T
    for got, ref in ((got_B, ref_B), (got_K, ref_K)):
        for c in range(4):
            assert np.abs(got[c] - ref[c]).max() < 1e-12 * max(1.0, np.abs(ref[c]).max()), c
    # a field without K tables reports K = 0
    GF0 = G.Field(_asym_field(with_K=False))
    K0, dK0 = GF0.kcov_eval(to_dev(s), to_dev(th), to_dev(ze))
    assert float(K0.abs().max()) == 0.0 and float(dK0.abs().max()) == 0.0


def test_tile_and_warp_kernels_refuse_fields_with_next4_tables():
    from paper_2605_16734_b200 import gcorbit as G
    GF = G.Field(_asym_field(M=8, N=8))
    for k in (G.GC_KERNEL_TILE, G.GC_KERNEL_WARP):
        with pytest.raises(G.GcError):
            GF.set_kernel(k)
    assert GF.kernel_info(100)["kernel"] == "generic" and GF.kernel_info(100_000)["kernel"] == "mma"


@pytest.mark.parametrize("with_K", [False, True])
@pytest.mark.parametrize("kernel", ["generic", "mma"])
def test_rhs_and_trace_with_sin_harmonics_and_K(kernel, with_K):
    """Right-hand side at 300 states (angles far from the origin, s spread over the grid) and a short trace of 300
    particles, both kernels that take such fields, against the oracle."""
    import torch
    import oracle
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld = _asym_field(with_K=with_K)
    spec = W.make_spec(0)
    P = W.make_particles(1, 300)
    OF, GF = oracle.OracleField(fld), G.Field(fld)
    mu = W.mu_from(P, OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    GF.set_kernel(dict(generic=G.GC_KERNEL_GENERIC, mma=G.GC_KERNEL_MMA)[kernel])
    assert GF.kernel_info(P.n)["kernel"] == kernel
    t = 1.7e-5
    y = np.stack([P.s, P.theta - 20.0, P.zeta + 70.0, P.vpar])
    got = GF.rhs_eval(spec.mass, spec.charge, t, to_dev(y), to_dev(mu))
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    ref = np.array([OF.rhs(spec.mass, spec.charge, mu[i], 1.0, t, y[:, i]) for i in range(P.n)]).T
    if with_K:                                                # K matters: the K = 0 equations give another answer
        ref0 = np.array([oracle.OracleField(_asym_field(with_K=False)).rhs(spec.mass, spec.charge, mu[i], 1.0, t, y[:, i])
                         for i in range(8)]).T
        assert np.abs(ref0[0] / ref[0, :8] - 1).max() > 1e-3
    for c in range(4):
        scale = np.maximum(np.abs(ref[c]), 1e-6 * np.abs(ref[c]).max())
        assert (np.abs(got[c] - ref[c]) / scale).max() < 1e-9, (c, (np.abs(got[c] - ref[c]) / scale).max())
    r = gpu_trace(GF, spec, P, mu, t_max=1.5e-5)
    o = OF.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=1.5e-5)
    cond = oracle_conditioning(OF, spec, P, mu, o, t_max=1.5e-5)
    info = assert_trace_parity(r, o, spec, label=f"next4 K={with_K} {kernel}", cond=cond, min_within=0.98)
    print(f"next4 K={with_K} {kernel}: {info}")


def test_full_launch_with_next4_tables_sampled():
    """20,000 particles through the mma kernel in its large-ensemble launch (full tiles, binning, parking), 64 of them
    against the oracle."""
    import oracle
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld = _asym_field()
    spec = W.make_spec(0)
    P = W.make_particles(1, 20_000)
    OF, GF = oracle.OracleField(fld), G.Field(fld)
    k = 64
    mu = W.mu_from(P, OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    assert GF.kernel_info(P.n)["kernel"] == "mma"
    r = gpu_trace(GF, spec, P, mu, t_max=1.0e-5)
    Q = P.head(k)
    o = OF.trace(spec, Q.s, Q.theta, Q.zeta, Q.vpar, mu[:k], t_max=1.0e-5)
    cond = oracle_conditioning(OF, spec, Q, mu[:k], o, t_max=1.0e-5)

    class Sub:
        y, t, status = r.y[:, :k], r.t[:k], r.status[:k]
        n_acc, n_rej, n_forced = r.n_acc[:k], r.n_rej[:k], r.n_forced[:k]
    info = assert_trace_parity(Sub, o, spec, label="next4 full launch mma", cond=cond, min_within=0.95, min_same=0.95)
    print(f"next4 full launch: {info}")
