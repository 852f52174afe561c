"""Shared helpers of the -m gpu parity tests: build both sides on the same seeded inputs and compare.

The CUDA path is always reached through the C ABI (paper_2605_16734_b200.gcorbit -> libgcorbit.so); the
expected values come from oracle/ only.  Tolerances:

* BASELINE.json north_star: final states within relative 1e-9 "over short horizons (before chaotic
  divergence)"; angles and s relative to max(1, |y|), v_par relative to max(v_ref, |v|).
* The adaptive controller on the C0 (piecewise-cubic) radial interpolant is itself an ill-conditioned map for a
  few particles: a 1-ulp change of theta0 moves the ORACLE's own end state by up to 1e-7 after 3000 steps
  (the step-size sequences drift apart by percents around rejected node crossings, and the two runs then differ
  by a fraction of the 1e-6 global truncation error).  No implementation can match the oracle more closely than
  the oracle matches itself, so each particle's tolerance is max(1e-9, COND_FACTOR * spread_i) where spread_i
  is measured from oracle runs alone (oracle_conditioning); the median over the ensemble must stay at
  rounding level, and the fraction of particles inside the flat 1e-9 is asserted per test.
* an accept/reject decision taken at err = 1 +- rounding can flip between two correct implementations; the
  fraction of particles whose (accepted, rejected) counts equal the oracle's is reported and bounded below.
"""
from __future__ import annotations

import numpy as np

SAME_RTOL = 1e-9
FLIP_RTOL = 1e-6
FLIP_FRACTION = 0.01
COND_FACTOR = 10.0
MEDIAN_RTOL = 1e-11


def to_dev(a, dtype=None):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=dtype or torch.float64, device="cuda:0")


def make_case(config: int, n: int | None = None, field=None):
    """(fld, spec, particles, oracle field, gpu field, mu) with mu from the oracle's B at the start point,
    the same array fed to both sides."""
    import oracle
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    fld = field if field is not None else W.make_field(config)
    spec = W.make_spec(config)
    P = W.make_particles(config, n)
    OF, GF = oracle.OracleField(fld), G.Field(fld)
    mu = W.mu_from(P, OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    return fld, spec, P, OF, GF, mu


def gpu_trace(GF, spec, P, mu, **kw):
    import torch
    from paper_2605_16734_b200 import gcorbit as G
    r = GF.trace(spec, to_dev(P.s), to_dev(P.theta), to_dev(P.zeta), to_dev(P.vpar), to_dev(mu), **kw)
    torch.cuda.synchronize()
    G.finish_poincare(r)
    return r


def rel_diff(y_gpu: np.ndarray, y_ref: np.ndarray, v_ref: float) -> np.ndarray:
    """[n] max over the four components of |gpu - ref| / max(|ref|, floor), floor = 1 for s, theta, zeta and
    v_ref for v_par."""
    floor = np.array([[1.0], [1.0], [1.0], [v_ref]])
    return (np.abs(y_gpu - y_ref) / np.maximum(np.abs(y_ref), floor)).max(axis=0)


def oracle_conditioning(OF, spec, P, mu, base, **kw):
    """Per-particle spread of the ORACLE's own result under ~1-ulp perturbations of theta0 and zeta0 (four
    extra oracle runs): (rel spread of y [n], rel spread of t_out [n], status stable [n])."""
    spread = np.zeros(P.n)
    tspread = np.zeros(P.n)
    stable = np.ones(P.n, bool)
    for a, b in [(1e-15, 0.0), (-1e-15, 0.0), (0.0, 1e-15), (0.0, -1e-15)]:
        o2 = OF.trace(spec, P.s, P.theta * (1.0 + a), P.zeta * (1.0 + b), P.vpar, mu, **kw)
        spread = np.maximum(spread, rel_diff(o2.y, base.y, spec.v_ref))
        tspread = np.maximum(tspread, np.abs(o2.t - base.t) / np.maximum(np.abs(base.t), 1e-300))
        stable &= o2.status == base.status
    return spread, tspread, stable


def assert_trace_parity(r_gpu, r_ref, spec, min_same=1.0 - FLIP_FRACTION, label="", cond=None,
                        min_within=1.0, median_rtol=MEDIAN_RTOL, flip_rtol=FLIP_RTOL):
    """cond = oracle_conditioning(...) or None (flat 1e-9 for particles on the oracle's step sequence,
    FLIP_RTOL for the others).  min_within: least fraction of particles inside the flat 1e-9."""
    yg = r_gpu.y.cpu().numpy()
    tg = r_gpu.t.cpu().numpy()
    stg = r_gpu.status.cpu().numpy()
    n = len(stg)
    if n == 0:
        return dict(same_frac=1.0, max_rel=0.0, within=1.0)
    stable = np.ones(n, bool) if cond is None else cond[2]
    bad = np.nonzero((stg != r_ref.status) & stable)[0]
    assert bad.size == 0, f"{label}: status differs at {bad[:8]}"
    same = (r_gpu.n_acc.cpu().numpy() == r_ref.n_acc) & (r_gpu.n_rej.cpu().numpy() == r_ref.n_rej)
    rel = rel_diff(yg, r_ref.y, spec.v_ref)
    relt = np.abs(tg - r_ref.t) / np.maximum(np.abs(r_ref.t), 1e-300)
    assert same.mean() >= min_same, f"{label}: only {same.mean() * 100:.2f} % of particles took the oracle's step sequence"
    assert np.median(rel) <= median_rtol, f"{label}: median rel diff {np.median(rel):.3e}"
    within = float((rel[stable] <= SAME_RTOL).mean())
    assert within >= min_within, f"{label}: only {within * 100:.2f} % of particles within {SAME_RTOL}"
    if cond is None:
        tol = np.where(same, SAME_RTOL, flip_rtol)
        tolt = np.where(same, SAME_RTOL, flip_rtol)
    else:
        # a flipped accept/reject decision puts the particle on another step sequence: bounded by FLIP_RTOL
        tol = np.where(same, np.maximum(SAME_RTOL, COND_FACTOR * cond[0]), flip_rtol)
        tolt = np.where(same, np.maximum(SAME_RTOL, COND_FACTOR * cond[1]), flip_rtol)
    worst = int(np.argmax(np.where(stable, rel / tol, 0.0)))
    assert (rel[stable] <= tol[stable]).all(), \
        f"{label}: particle {worst}: rel diff {rel[worst]:.3e} > tolerance {tol[worst]:.3e}"
    assert (relt[stable] <= tolt[stable]).all(), f"{label}: t_out differs by {relt[stable].max():.3e}"
    assert rel[stable].max() <= flip_rtol, f"{label}: max rel diff {rel.max():.3e} > {flip_rtol}"
    if same.any():
        assert np.array_equal(r_gpu.n_forced.cpu().numpy()[same], r_ref.n_forced[same])
    info = dict(same_frac=float(same.mean()), max_rel=float(rel[stable].max()), median_rel=float(np.median(rel)),
                within=within, max_rel_t=float(relt[stable].max()))
    record_info("trace_parity", label=label, particles=int(n), unstable_in_oracle=int((~stable).sum()), **info)
    return info


def record_info(kind: str, **kw):
    """Append one JSON line per comparison to gpurun_out/parity_info.jsonl (scratch that comes back from the GPU box;
    profiles/r2_parity_summary.md is assembled from it), so that how close each test got is on record."""
    import json
    import os
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    if os.path.isdir(out):
        test = os.environ.get("PYTEST_CURRENT_TEST", "").split(" ")[0]
        with open(os.path.join(out, "parity_info.jsonl"), "a") as fh:
            fh.write(json.dumps(dict(kind=kind, test=test, **kw)) + "\n")


def sort_poincare(rec: np.ndarray) -> np.ndarray:
    rec = np.asarray(rec)
    if rec.shape[0] == 0:
        return rec
    return rec[np.lexsort((rec[:, 1], rec[:, 0]))]
