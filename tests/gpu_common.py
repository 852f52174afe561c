"""Shared helpers of the -m gpu parity tests: build both sides on the same seeded inputs and compare.

The CUDA path is always reached through the C ABI (paper_2605_16734_b200.gcorbit -> libgcorbit.so); the
expected values come from oracle/ only.  Tolerances:

* a particle whose accepted / rejected step counts equal the oracle's took the same step sequence; its final
  state must agree to relative 1e-9 (BASELINE.json north_star; angles and s relative to max(1, |y|), v_par
  relative to max(v_ref, |v|));
* an accept/reject decision taken at err = 1 +- rounding can flip between two correct implementations; from
  there on the two step sequences differ and the states agree to the integrator's own global error, not
  to rounding.  Such particles must stay below FLIP_FRACTION of the ensemble and within FLIP_RTOL.
"""
from __future__ import annotations

import numpy as np

SAME_RTOL = 1e-9
FLIP_RTOL = 1e-6
FLIP_FRACTION = 0.01


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


def assert_trace_parity(r_gpu, r_ref, spec, min_same=1.0 - FLIP_FRACTION, label=""):
    yg = r_gpu.y.cpu().numpy()
    tg = r_gpu.t.cpu().numpy()
    stg = r_gpu.status.cpu().numpy()
    assert np.array_equal(stg, r_ref.status), f"{label}: status differs at {np.nonzero(stg != r_ref.status)[0][:8]}"
    same = (r_gpu.n_acc.cpu().numpy() == r_ref.n_acc) & (r_gpu.n_rej.cpu().numpy() == r_ref.n_rej)
    rel = rel_diff(yg, r_ref.y, spec.v_ref)
    n = len(rel)
    if n == 0:
        return dict(same_frac=1.0, max_rel_same=0.0, max_rel=0.0)
    assert same.mean() >= min_same, f"{label}: only {same.mean() * 100:.2f} % of particles took the oracle's step sequence"
    if same.any():
        assert rel[same].max() <= SAME_RTOL, f"{label}: max rel diff {rel[same].max():.3e} > {SAME_RTOL} (same step sequence)"
        dt = np.abs(tg - r_ref.t)[same]
        assert (dt <= 1e-12 * np.maximum(np.abs(r_ref.t[same]), 1e-30) + 1e-300).all(), f"{label}: t_out differs"
        assert np.array_equal(r_gpu.n_forced.cpu().numpy()[same], r_ref.n_forced[same])
    assert rel.max() <= FLIP_RTOL, f"{label}: max rel diff {rel.max():.3e} > {FLIP_RTOL}"
    return dict(same_frac=float(same.mean()), max_rel_same=float(rel[same].max()) if same.any() else 0.0,
                max_rel=float(rel.max()))


def sort_poincare(rec: np.ndarray) -> np.ndarray:
    rec = np.asarray(rec)
    if rec.shape[0] == 0:
        return rec
    return rec[np.lexsort((rec[:, 1], rec[:, 0]))]
