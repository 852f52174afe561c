"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the seeded
synthetic inputs of BASELINE.json:configs (SURVEY.md section 8(c) "GPU-vs-oracle acceptance")."""
from __future__ import annotations

import numpy as np
import pytest

from gpu_common import (COND_FACTOR, FLIP_RTOL, SAME_RTOL, assert_trace_parity, gpu_trace, make_case,
                        oracle_conditioning, rel_diff, sort_poincare, to_dev)

pytestmark = pytest.mark.gpu

KERNELS = ["generic", "warp", "tile", "mma"]


def _set_kernel(GF, name):
    from paper_2605_16734_b200 import gcorbit as G
    GF.set_kernel({"generic": G.GC_KERNEL_GENERIC, "warp": G.GC_KERNEL_WARP, "tile": G.GC_KERNEL_TILE, "mma": G.GC_KERNEL_MMA,
                   "auto": G.GC_KERNEL_AUTO}[name])


@pytest.fixture(scope="module")
def cases():
    cache = {}

    def get(config, n):
        if (config, n) not in cache:
            cache[(config, n)] = make_case(config, n)
        return cache[(config, n)]
    return get


# ---- O2 / O3: point evaluations ---------------------------------------------------------------------------------
@pytest.mark.parametrize("config", [0, 1])
def test_field_eval_matches_oracle(cases, config):
    import torch
    fld, spec, P, OF, GF, mu = cases(config, 300)
    # include points outside [0, 1] (clamped stencil extrapolates, A6) and large unwrapped angles (A12)
    s = P.s.copy(); th = P.theta.copy(); ze = P.zeta.copy()
    s[:4] = [-0.01, 0.0, 1.0, 1.02]
    th[4:8] += 5.0e3
    ze[8:12] -= 2.0e4
    B, dB = GF.field_eval(to_dev(s), to_dev(th), to_dev(ze))
    torch.cuda.synchronize()
    ref = OF.eval_B_many(s, th, ze)
    B, dB = B.cpu().numpy(), dB.cpu().numpy()
    assert np.abs(B / ref[:, 0] - 1.0).max() < 1e-12
    for c in range(3):
        # unwrapped angles of 1e4 rad carry 1e4 * eps of phase noise on BOTH sides
        assert np.abs(dB[c] - ref[:, 1 + c]).max() <= 1e-10 * np.abs(ref[:, 1 + c]).max()


@pytest.mark.parametrize("config", [2, 4])
def test_pert_eval_matches_oracle(cases, config):
    import torch
    fld, spec, P, OF, GF, mu = cases(config, 200)
    t = 3.7e-5
    out = GF.pert_eval(to_dev(P.s), to_dev(P.theta), to_dev(P.zeta), t)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    ref = np.array([OF.eval_pert(P.s[i], P.theta[i], P.zeta[i], t) for i in range(P.n)]).T
    for q in range(9):
        assert np.abs(out[q] - ref[q]).max() <= 1e-11 * np.abs(ref[q]).max(), q


def test_pert_eval_static_field_is_zero(cases):
    import torch
    fld, spec, P, OF, GF, mu = cases(0, 64)
    out = GF.pert_eval(to_dev(P.s), to_dev(P.theta), to_dev(P.zeta), 1e-5)
    torch.cuda.synchronize()
    assert float(out.abs().max()) == 0.0


# ---- O4: the right-hand side alone, both kernels ------------------------------------------------------------------
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("config", [0, 1, 2, 4])
def test_rhs_matches_oracle(cases, config, kernel):
    import torch
    fld, spec, P, OF, GF, mu = cases(config, 256)
    _set_kernel(GF, kernel)
    t = 3.3e-5
    y = np.stack([P.s, P.theta + 50.0, P.zeta - 30.0, P.vpar])
    got = GF.rhs_eval(spec.mass, spec.charge, t, to_dev(y), to_dev(mu))
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    ref = np.array([OF.rhs(spec.mass, spec.charge, mu[i], 1.0, t, y[:, i]) for i in range(P.n)]).T
    for c in range(4):
        scale = np.maximum(np.abs(ref[c]), 1e-6 * np.abs(ref[c]).max())
        assert (np.abs(got[c] - ref[c]) / scale).max() < 1e-9, (c, (np.abs(got[c] - ref[c]) / scale).max())
    _set_kernel(GF, "auto")


# ---- O5-O7: the trace ---------------------------------------------------------------------------------------------
_FULL = {}


def _oracle_full(cases):
    """Config 0 oracle run and its conditioning, computed once for both kernels."""
    if not _FULL:
        fld, spec, P, OF, GF, mu = cases(0, None)
        o = OF.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu)
        _FULL["o"], _FULL["cond"] = o, oracle_conditioning(OF, spec, P, mu, o)
    return _FULL["o"], _FULL["cond"]


@pytest.mark.parametrize("kernel", KERNELS)
def test_trace_config0_full(cases, kernel):
    """BASELINE.json configs[0] in full: 512 alphas, t_max = 1e-4 s, rtol 1e-9."""
    fld, spec, P, OF, GF, mu = cases(0, None)
    assert P.n == 512 and spec.t_max == 1e-4
    _set_kernel(GF, kernel)
    r = gpu_trace(GF, spec, P, mu)
    o, cond = _oracle_full(cases)
    # 1e-4 s is ~3000 steps: ~1-2 % of the particles are ill-conditioned in the oracle itself (gpu_common)
    info = assert_trace_parity(r, o, spec, label=f"config 0 {kernel}", cond=cond, min_within=0.95)
    print(f"config 0 {kernel}: {info}, attempts {int(o.n_acc.sum() + o.n_rej.sum())}")
    _set_kernel(GF, "auto")


_SHORT = {}


@pytest.mark.parametrize("kernel", KERNELS)
def test_trace_config0_flat_1e9(cases, kernel):
    """BASELINE.json north_star, to the letter: "final states within relative 1e-9 over short horizons (before chaotic
    divergence)".  Config 0, all 512 particles, t_max = 2e-5 s (~600 attempted steps): at this horizon the oracle
    reproduces ITSELF to 1.1e-10 under 1-ulp changes of the start angles (VERDICT round 2, weak point 2), so the flat
    rule can hold for every particle and is asserted for every particle: no per-particle conditioning, no
    flipped-decision allowance on the states (min_within = 1.0)."""
    fld, spec, P, OF, GF, mu = cases(0, None)
    assert P.n == 512
    _set_kernel(GF, kernel)
    r = gpu_trace(GF, spec, P, mu, t_max=2e-5)
    _set_kernel(GF, "auto")
    if "o" not in _SHORT:
        _SHORT["o"] = OF.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=2e-5)
    info = assert_trace_parity(r, _SHORT["o"], spec, label=f"config 0 flat 1e-9 {kernel}", cond=None, min_within=1.0)
    assert info["max_rel"] <= SAME_RTOL and info["max_rel_t"] <= SAME_RTOL
    print(f"config 0 flat {kernel}: {info}")


_SUB = {}


@pytest.mark.parametrize("kernel", ["warp", "tile", "mma"])
@pytest.mark.parametrize("config,n,t_max", [(1, 296, 2e-5), (2, 256, 2e-5), (3, 301, 3e-5), (4, 256, 2e-5)])
def test_trace_subsamples(cases, config, n, t_max, kernel):
    """Short-horizon subsamples of configs 1-4 (n chosen ragged against 8 warps per block and 128-particle
    tiles), hot-path kernels."""
    fld, spec, P, OF, GF, mu = cases(config, n)
    cap = 4096 if config == 4 else 0
    _set_kernel(GF, kernel)
    r = gpu_trace(GF, spec, P, mu, t_max=t_max, poincare_capacity=cap)
    _set_kernel(GF, "auto")
    if config not in _SUB:
        o = OF.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=t_max, poincare_capacity=cap)
        _SUB[config] = (o, oracle_conditioning(OF, spec, P, mu, o, t_max=t_max))
    o, cond = _SUB[config]
    info = assert_trace_parity(r, o, spec, label=f"config {config} {kernel}", cond=cond, min_within=0.99)
    print(f"config {config}: {info}")
    if cap:
        # O8: same crossings (record order is unspecified: compare sorted by particle, time)
        assert r.poincare_count == o.poincare_count > 0
        a, b = sort_poincare(r.poincare.cpu().numpy()), sort_poincare(o.poincare)
        assert np.array_equal(a[:, 0], b[:, 0])
        assert np.abs(a[:, 1] - b[:, 1]).max() <= 1e-9 * t_max
        assert np.abs(a[:, 2] - b[:, 2]).max() <= 1e-9
        dth = np.abs(a[:, 3] - b[:, 3])
        assert np.minimum(dth, 2 * np.pi - dth).max() <= 1e-8


def test_trace_generic_kernel_with_modes(cases):
    fld, spec, P, OF, GF, mu = cases(2, 256)
    _set_kernel(GF, "generic")
    r = gpu_trace(GF, spec, P.head(64), mu[:64], t_max=1e-5)
    Q = P.head(64)
    o = OF.trace(spec, Q.s, Q.theta, Q.zeta, Q.vpar, mu[:64], t_max=1e-5)
    cond = oracle_conditioning(OF, spec, Q, mu[:64], o, t_max=1e-5)
    assert_trace_parity(r, o, spec, min_same=0.95, label="config 2 generic", cond=cond, min_within=0.98)
    _set_kernel(GF, "auto")


@pytest.mark.parametrize("kernel", ["warp", "tile", "mma"])
@pytest.mark.parametrize("n", [1, 7, 33, 148 * 8 + 3])
def test_trace_ragged_sizes(cases, n, kernel):
    """One particle, fewer particles than warps in a block / lanes in a tile, and one more wave than the
    persistent grid holds."""
    fld, spec, P, OF, GF, mu = cases(0, 148 * 8 + 3)
    Q = P.head(n)
    _set_kernel(GF, kernel)
    r = gpu_trace(GF, spec, Q, mu[:n], t_max=3e-6)
    _set_kernel(GF, "auto")
    o = OF.trace(spec, Q.s, Q.theta, Q.zeta, Q.vpar, mu[:n], t_max=3e-6)
    cond = oracle_conditioning(OF, spec, Q, mu[:n], o, t_max=3e-6)
    assert_trace_parity(r, o, spec, min_same=0.0 if n < 100 else 0.99, label=f"n={n}", cond=cond)


@pytest.mark.parametrize("config,n_full,seg", [(1, 100_000, 2e-5), (2, 100_000, 2e-5), (3, 1_000_000, 4e-6),
                                               (4, 1_000_000, 4e-6)])
def test_full_size_launch_sampled(cases, config, n_full, seg):
    """BASELINE.json configs[1], [2], [3] and [4] at FULL size in the launch configuration bench.py times (100,000
    particles over 2e-5 s segments; 10^6 particles, shorter segments to keep the test short), in-place resume of a
    second segment; 48 sampled particles (and a few lost ones) checked one by one against the oracle."""
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    fld, spec, P, OF, GF, _ = cases(config, 64)     # fields only; the full ensemble is drawn here
    assert GF.kernel_info(n_full)["kernel"] == "mma"
    from paper_2605_16734_b200 import workloads as W
    P = W.make_particles(config)
    assert P.n == n_full
    s, th, ze, vp = (to_dev(x) for x in (P.s, P.theta, P.zeta, P.vpar))
    B, _ = GF.field_eval(s, th, ze, derivs=False)
    mu_d = to_dev(0.5 * spec.mass * P.vperp2()) / B
    h = torch.zeros(P.n, dtype=torch.float64, device="cuda:0")
    st = GF.trace(spec, s, th, ze, vp, mu_d, h_inout=h, t0=0.0, t_max=seg)
    GF.trace_resume(spec, st, mu_d, t0=seg, t_max=2 * seg)
    torch.cuda.synchronize()
    status = st.status.cpu().numpy()
    assert set(np.unique(status)) <= {0, 1, 2}
    assert (st.t.cpu().numpy()[status == 0] == 2 * seg).all()
    idx = np.random.default_rng(7).choice(P.n, 48, replace=False)
    idx = np.union1d(idx, np.nonzero(status == 1)[0][:8])          # and a few lost ones if any
    mu = mu_d.cpu().numpy()
    Q = W.Particles(P.s[idx], P.theta[idx], P.zeta[idx], P.pitch[idx], P.speed[idx])

    def two_segments(Qp):
        o1 = OF.trace(spec, Qp.s, Qp.theta, Qp.zeta, Qp.vpar, mu[idx], t0=0.0, t_max=seg)
        alive = o1.status == 0
        o2 = OF.trace(spec, o1.y[0, alive], o1.y[1, alive], o1.y[2, alive], o1.y[3, alive], mu[idx][alive],
                      h_in=o1.h[alive], t0=seg, t_max=2 * seg)
        y_ref, st_ref, t_ref = o1.y.copy(), o1.status.copy(), o1.t.copy()
        y_ref[:, alive], st_ref[alive], t_ref[alive] = o2.y, o2.status, o2.t
        two_segments.counts = (o1.n_acc.copy(), o1.n_rej.copy())
        two_segments.counts[0][alive] += o2.n_acc
        two_segments.counts[1][alive] += o2.n_rej
        return y_ref, st_ref, t_ref

    y_ref, st_ref, t_ref = two_segments(Q)
    acc_ref, rej_ref = two_segments.counts
    # the oracle's own conditioning on these particles (gpu_common): theta0 moved by ~1 ulp
    spread, tspread = np.zeros(len(idx)), np.zeros(len(idx))
    for a, b in [(1e-15, 0.0), (-1e-15, 0.0), (0.0, 1e-15), (0.0, -1e-15)]:     # as gpu_common.oracle_conditioning
        Qp = W.Particles(Q.s, Q.theta * (1.0 + a), Q.zeta * (1.0 + b), Q.pitch, Q.speed)
        y2, st2, t2 = two_segments(Qp)
        assert np.array_equal(st2, st_ref)
        spread = np.maximum(spread, rel_diff(y2, y_ref, spec.v_ref))
        tspread = np.maximum(tspread, np.abs(t2 - t_ref) / t_ref)
    assert np.array_equal(status[idx], st_ref)
    rel = rel_diff(st.y.cpu().numpy()[:, idx], y_ref, spec.v_ref)
    # DESIGN.md section 5 ("Controller decisions"), the rule assert_trace_parity applies: a particle on the oracle's
    # step sequence is held to max(1e-9, 10 x the oracle's own spread); an accept/reject decision taken at
    # err = 1 +- 1e-13 may flip, the two step sequences then differ and the results agree to the truncation error
    # only (FLIP_RTOL); at most 5 % of the sampled particles may do that
    same = (st.n_acc.cpu().numpy()[idx] == acc_ref) & (st.n_rej.cpu().numpy()[idx] == rej_ref)
    assert same.mean() >= 0.95, same.mean()
    tol = np.where(same, np.maximum(SAME_RTOL, COND_FACTOR * spread), FLIP_RTOL)
    assert np.median(rel) < 1e-11 and (rel <= tol).all(), (rel.max(), np.nonzero(rel > tol)[0])
    relt = np.abs(st.t.cpu().numpy()[idx] - t_ref) / t_ref
    assert (relt <= np.where(same, np.maximum(SAME_RTOL, COND_FACTOR * tspread), FLIP_RTOL)).all(), relt.max()
    from gpu_common import record_info
    record_info("full_size_sampled", label=f"config {config} mma, {n_full} particles, 2 x {seg:g} s", particles=len(idx),
                max_rel=float(rel.max()), median_rel=float(np.median(rel)), within=float((rel <= SAME_RTOL).mean()),
                max_rel_t=float(relt.max()), same_frac=float(same.mean()), waves=-(-n_full // (1 << 18)))


@pytest.mark.parametrize("kernel", ["tile", "mma"])
def test_trace_fine_grid_steps_across_several_cells(kernel):
    """A radial grid so fine (ns = 801) and a tolerance so loose (1e-4) that single steps cross more than a
    cell: stage points land outside the staged window and particles are parked and re-binned all the time, which
    exercises the global-memory sweep and the parking of the cell-binned kernels.  10,000 particles traced
    (fills tiles and groups), 200 of them checked one by one."""
    import dataclasses
    import oracle
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld = W.make_equilibrium(16, 16, 801)
    spec = dataclasses.replace(W.make_spec(0), rtol=1e-4, atol=1e-4, t_max=6e-6)
    P = W.make_particles(1, 10_000)
    OF, GF = oracle.OracleField(fld), G.Field(fld)
    k = 200
    mu = W.mu_from(P, OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    _set_kernel(GF, kernel)
    assert GF.kernel_info(P.n)["kernel"] == kernel
    r = gpu_trace(GF, spec, P, mu)
    Q = P.head(k)
    o = OF.trace(spec, Q.s, Q.theta, Q.zeta, Q.vpar, mu[:k])
    ds = np.abs(o.y[0] - Q.s) * (fld.ns - 1)
    assert ds.max() > 8.0, "the case is meant to carry particles across many cells"
    cond = oracle_conditioning(OF, spec, Q, mu[:k], o)
    # the 1-ulp input perturbations of oracle_conditioning do not reach the cancellation noise of B_s (below), which
    # accumulates to ~1e-9..1e-8 over the ~600 right-hand sides of this run: floor the per-particle spread at 1e-8
    # (tolerance 1e-7; a wrong row or weight in the fallback sweep shows up at >= 1e-3)
    cond = (np.maximum(cond[0], 1e-8), np.maximum(cond[1], 1e-8), cond[2])

    class Sub:                      # the first k particles of the GPU result
        y, t, status = r.y[:, :k], r.t[:k], r.status[:k]
        n_acc, n_rej, n_forced = r.n_acc[:k], r.n_rej[:k], r.n_forced[:k]
    # d/ds weights carry the factor ns - 1 = 800: sum_a dw_a T_a cancels 800 x 5.7 T down to |B_s| ~ 0.1 T, which
    # costs three to four more digits than on the 101-node grids of the configs, on BOTH sides (the oracle's own
    # spread under 1-ulp input changes shows it).  So the median bound is 1e-9 here instead of 1e-11, the flat
    # 1e-9 must hold for half of the particles only, and every particle on the oracle's step sequence is held to 10 x the oracle's own spread (the <= 3 % with a
    # flipped accept/reject decision to 1e3 x rtol: at rtol = 1e-4 a different step sequence costs ~1e-2).
    info = assert_trace_parity(Sub, o, spec, label=f"fine grid {kernel}", cond=cond, min_same=0.97, min_within=0.5,
                               median_rtol=1e-9, flip_rtol=1e3 * spec.rtol)
    print(f"fine grid {kernel}: {info}, cells crossed up to {ds.max():.1f}")


@pytest.mark.parametrize("kernel", KERNELS)
def test_general_field_rhs_and_trace(kernel):
    """A field that exercises what the configs leave at zero: I(s) != 0, G'(s) != 0, nonlinear iota, harmonics given
    in shuffled order with a duplicated (m, n) pair (duplicates add, gcorbit.h), M = 11 and N = 13 (zero-padded in the
    packed layouts), two modes with different omega.  Right-hand side at 300 points and a short trace of 300
    particles against the oracle, every kernel."""
    import torch
    import oracle
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    rng = np.random.default_rng(5)
    ns, nfp, M, N = 61, 3, 11, 13
    xm, xn = W.harmonic_list(M, N)
    s_n = np.arange(ns) / (ns - 1)
    amp = 0.04 * 5.0 * rng.standard_normal(xm.size) * np.exp(-(xm + np.abs(xn)) / 3.0)
    bmnc = amp[None, :] * (s_n[:, None] ** (xm[None, :] / 2.0))
    bmnc[:, 0] = 5.0 + 0.3 * s_n
    perm = rng.permutation(xm.size)
    xm, xn, bmnc = xm[perm], xn[perm], bmnc[:, perm]
    dup = int(np.nonzero((xm == 3) & (xn == -2))[0][0])
    xm, xn = np.append(xm, xm[dup]), np.append(xn, xn[dup])               # the same harmonic once more: adds
    bmnc = np.concatenate([bmnc, 0.5 * bmnc[:, dup:dup + 1]], axis=1)
    env = np.exp(-(s_n - 0.45) ** 2 / (2 * 0.08 ** 2))
    fld = W.Field(ns=ns, nfp=nfp, xm=xm.astype(np.int32), xn=xn.astype(np.int32), bmnc=np.ascontiguousarray(bmnc),
                  G=48.0 + 2.0 * s_n - 0.7 * s_n ** 2, I=1.5 * s_n + 0.4 * s_n ** 2,
                  iota=0.38 + 0.2 * s_n - 0.05 * s_n ** 3, psi0=6.5,
                  mode_m=np.array([4, 7], np.int32), mode_n=np.array([-3, 5], np.int32),
                  mode_omega=2 * np.pi * np.array([90e3, -210e3]), mode_phase=np.array([0.4, 2.0]),
                  phihat=np.stack([3e3 * env, -2e3 * env], axis=1))
    spec = W.make_spec(0)
    P = W.make_particles(1, 300)
    OF, GF = oracle.OracleField(fld), G.Field(fld)
    mu = W.mu_from(P, OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    _set_kernel(GF, kernel)
    t = 1.7e-5
    y = np.stack([P.s, P.theta - 20.0, P.zeta + 70.0, P.vpar])
    got = GF.rhs_eval(spec.mass, spec.charge, t, to_dev(y), to_dev(mu))
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    ref = np.array([OF.rhs(spec.mass, spec.charge, mu[i], 1.0, t, y[:, i]) for i in range(P.n)]).T
    for c in range(4):
        scale = np.maximum(np.abs(ref[c]), 1e-6 * np.abs(ref[c]).max())
        assert (np.abs(got[c] - ref[c]) / scale).max() < 1e-9, (c, (np.abs(got[c] - ref[c]) / scale).max())
    r = gpu_trace(GF, spec, P, mu, t_max=1.5e-5)
    o = OF.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=1.5e-5)
    cond = oracle_conditioning(OF, spec, P, mu, o, t_max=1.5e-5)
    info = assert_trace_parity(r, o, spec, label=f"general field {kernel}", cond=cond, min_within=0.98)
    print(f"general field {kernel}: {info}")
