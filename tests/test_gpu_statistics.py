"""-m gpu: ensemble statistics over a horizon long enough for losses (BASELINE.json north_star: "Ensemble loss
fractions must agree within the Monte Carlo standard error, with loss-time histograms passing a two-sample KS
test at p>0.01"; the paper's two-code comparison PAPER.md:68,72).

Expected values: tests/golden/statistics_config{1,2,3,4}.txt, ORACLE ensembles of 2048 particles traced to 1e-3 s,
written by tests/golden/make_statistics_golden.py (oracle/ only), the size SURVEY.md section 8(d) asks for.  For each
of the four configurations with losses the CUDA path traces (a) the same 2048 particles (small-ensemble kernel and the
large-ensemble mma kernel) and (b) an independent draw of 100,000 particles of the same recipe (mma kernel).
Config 0 loses nothing inside its 1e-4 s horizon and is compared particle by particle in test_gpu_parity.py."""
from __future__ import annotations

import json
import os

import numpy as np
import pytest

from gpu_common import gpu_trace, make_case, to_dev

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))
T_MAX = 1e-3
N_ORACLE = 2048
N_INDEPENDENT = 100_000


def _golden(config):
    path = os.path.join(HERE, "golden", f"statistics_config{config}.txt")
    if not os.path.exists(path):
        pytest.fail(f"{path} missing: run python tests/golden/make_statistics_golden.py --configs {config}")
    a = np.loadtxt(path)
    assert a.shape == (N_ORACLE, 4)
    return a[:, 0].astype(int), a[:, 1], a[:, 2]


def _loss(status, t):
    status, t = np.asarray(status), np.asarray(t)
    return float((status == 1).mean()), np.sort(t[status == 1])


def _record(name, **kw):
    out = os.path.join(os.path.dirname(HERE), "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "statistics_info.jsonl"), "a") as fh:
            fh.write(json.dumps(dict(test=name, **kw)) + "\n")


@pytest.mark.parametrize("config", [1, 2, 3, 4])
def test_loss_fraction_and_loss_times_against_the_oracle_ensemble(config):
    import torch
    from scipy.stats import ks_2samp
    from paper_2605_16734_b200 import gcorbit as G, workloads as W
    st_o, t_o, s_o = _golden(config)
    f_o, lt_o = _loss(st_o, t_o)
    assert len(lt_o) >= 100, "horizon too short for a loss statistic"
    fld, spec, P, OF, GF, mu = make_case(config, N_ORACLE)

    # (a) the same ensemble: loss fraction within 2 sqrt(f (1 - f) 2 / N) (SURVEY.md 8(c) acceptance), KS p > 0.01
    se = 2.0 * np.sqrt(f_o * (1 - f_o) * 2.0 / N_ORACLE)
    info = dict(config=config, oracle_loss_fraction=f_o, oracle_axis_fraction=float((st_o == 2).mean()),
                loss_events=len(lt_o), bound_same=se)
    for name, kern in (("auto", G.GC_KERNEL_AUTO), ("mma", G.GC_KERNEL_MMA)):
        GF.set_kernel(kern)
        g = gpu_trace(GF, spec, P, mu, t_max=T_MAX)
        st, t = g.status.cpu().numpy(), g.t.cpu().numpy()
        f_g, lt_g = _loss(st, t)
        p = ks_2samp(lt_g, lt_o).pvalue
        info[name] = dict(kernel=GF.kernel_info(P.n)["kernel"], loss_fraction=f_g, ks_p=float(p),
                          axis_fraction=float((st == 2).mean()), status_equal=float((st == st_o).mean()))
        # the SAME particles on the SAME field and integrator: the paired comparison is the sharp one (the two-sample
        # Monte Carlo bound below would let 2.5 % of the ensemble change sides) -- measured 100 %
        assert (st == st_o).mean() >= 0.98, (name, float((st == st_o).mean()))
        assert abs(f_g - f_o) <= se, (name, f_g, f_o, se)
        assert p > 0.01, (name, p)
        assert set(np.unique(st)) <= {0, 1, 2}              # no particle ends in a state the config cannot produce
        assert abs((st == 2).mean() - (st_o == 2).mean()) <= se
        # survivors sit exactly at t_max; lost particles report the end of the step that crossed s = 1 (O7)
        y = g.y.cpu().numpy()
        assert (t[st == 0] == T_MAX).all() and (t[st == 1] < T_MAX).all()
        assert (y[0, st == 1] >= spec.s_loss).all() and (y[0, st == 0] < spec.s_loss).all()
    GF.set_kernel(G.GC_KERNEL_AUTO)

    # (b) an independent, fifty times larger draw of the same recipe through the large-ensemble kernel
    P2 = W.make_particles(config, N_INDEPENDENT, stream=5)
    s, th, ze = to_dev(P2.s), to_dev(P2.theta), to_dev(P2.zeta)
    B, _ = GF.field_eval(s, th, ze, derivs=False)
    mu2 = to_dev(0.5 * spec.mass * P2.vperp2()) / B
    assert GF.kernel_info(P2.n)["kernel"] == "mma"
    g2 = GF.trace(spec, s, th, ze, to_dev(P2.vpar), mu2, t_max=T_MAX)
    torch.cuda.synchronize()
    st2, t2 = g2.status.cpu().numpy(), g2.t.cpu().numpy()
    f_2, lt_2 = _loss(st2, t2)
    se2 = 3.0 * np.sqrt(f_o * (1 - f_o) / N_ORACLE + f_2 * (1 - f_2) / N_INDEPENDENT)
    p2 = ks_2samp(lt_2, lt_o).pvalue
    info["independent"] = dict(particles=N_INDEPENDENT, loss_fraction=f_2, ks_p=float(p2), bound=se2,
                               axis_fraction=float((st2 == 2).mean()))
    _record("loss_statistics", **info)
    print(json.dumps(info))
    assert abs(f_2 - f_o) <= se2, (f_2, f_o, se2)
    assert p2 > 0.01, p2
    assert set(np.unique(st2)) <= {0, 1, 2}


def test_energy_conserved_on_gpu():
    """Check (a) of SURVEY.md section 8(c) applied to the CUDA path itself: E = m v_par^2 / 2 + mu B is
    conserved by the static-field equations, so the GPU end states must keep it to ~steps * rtol."""
    import torch
    fld, spec, P, OF, GF, mu = make_case(0, None)
    r = gpu_trace(GF, spec, P, mu)
    y = r.y
    B1, _ = GF.field_eval(y[0].contiguous(), y[1].contiguous(), y[2].contiguous(), derivs=False)
    torch.cuda.synchronize()
    E0 = 0.5 * spec.mass * P.vpar ** 2 + mu * OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0]
    E1 = 0.5 * spec.mass * y[3].cpu().numpy() ** 2 + mu * B1.cpu().numpy()
    ok = r.status.cpu().numpy() == 0
    drift = np.abs(E1 / E0 - 1.0)[ok]
    # each accepted step may add up to ~rtol of relative energy error; the oracle's own drift on this
    # ensemble peaks at 1.6e-7 (3000 steps at rtol 1e-9)
    steps = r.n_acc.cpu().numpy()[ok]
    assert (drift <= 1e-9 * steps).all() and drift.max() < 1e-6, drift.max()


@pytest.mark.parametrize("kind", ["lagrange", "hermite"])
@pytest.mark.parametrize("config", [1, 3])
def test_interpolant_ensembles_reproduce_the_direct_sum_loss_statistics(config, kind):
    """NEXT-2 as a replacement for the direct sum: the SAME 2048 particles traced to 1e-3 s on the tricubic interpolant
    (101 x 128 x 128 nodes, either reading) against the DIRECT-SUM oracle ensemble -- a different field representation
    (interpolation error ~1e-6 of B), so single orbits differ after a few bounce times, but the ensemble loss fraction
    must agree within the Monte Carlo standard error and the loss times pass the KS test, as between two codes
    ("two codes report identical loss fractions").

    What this does NOT show: at N = 2048 the Monte Carlo bound is +-0.02, so the test has no power against a bias of a
    few 1e-3.  The full-size run (profiles/r2_full_runs.md: config 3, 10^6 particles to 2e-2 s) gives 0.1988 on the
    Hermite 101 x 128 x 128 interpolant against 0.1946 on the direct sum, about 7 standard errors at that size: that
    grid at rtol 1e-8 does NOT meet north_star's loss-fraction criterion on the target configuration, and its speed is
    quoted as that of a reduced-accuracy field (README).  The sharper statement this test can
    make at its size is the paired one: at 1e-3 s at most 3 % of the same particles end differently (measured
    0.1-1.5 %)."""
    from scipy.stats import ks_2samp
    from paper_2605_16734_b200 import gcorbit as G
    st_o, t_o, s_o = _golden(config)
    f_o, lt_o = _loss(st_o, t_o)
    fld, spec, P, OF, GF, mu = make_case(config, N_ORACLE)
    GF.set_grid(101, 128, 128, kind=G.GC_GRID_HERMITE if kind == "hermite" else G.GC_GRID_LAGRANGE)
    assert GF.kernel_info(P.n)["kernel"] == "grid"
    g = gpu_trace(GF, spec, P, mu, t_max=T_MAX)                 # mu from the direct-sum B at the start points
    st, t = g.status.cpu().numpy(), g.t.cpu().numpy()
    f_g, lt_g = _loss(st, t)
    se = 2.0 * np.sqrt(f_o * (1 - f_o) * 2.0 / N_ORACLE)
    p = ks_2samp(lt_g, lt_o).pvalue
    attempts = int(g.n_acc.sum().item() + g.n_rej.sum().item())
    _record("interpolant_loss_statistics", config=config, kind=kind, oracle_loss_fraction=f_o, loss_fraction=f_g,
            bound=se, ks_p=float(p), status_equal=float((st == st_o).mean()), attempts=attempts,
            accepted_fraction=float(g.n_acc.sum().item()) / attempts)
    assert (st == st_o).mean() >= 0.97, float((st == st_o).mean())
    assert abs(f_g - f_o) <= se, (f_g, f_o, se)
    assert p > 0.01, p
    assert set(np.unique(st)) <= {0, 1, 2}


@pytest.mark.parametrize("field", ["sum", "hermite"])
@pytest.mark.parametrize("config", [1, 3])
def test_symplectic_ensembles_reproduce_the_dormand_prince_loss_statistics(config, field):
    """The paper's cross-code comparison (an adaptive Runge-Kutta code against a symplectic one, "the
    two codes report identical loss fractions") inside this library: the SAME 2048 particles advanced to 1e-3 s by
    gc_trace_symplectic (dt = 2e-8 s, 50,000 steps) on the direct sum and on the Hermite interpolant against the
    Dormand-Prince ORACLE ensemble.  A first-order scheme at this step follows single orbits to ~1e-2 only, so what
    must agree is the ensemble: loss fraction within the Monte Carlo standard error, KS on the loss times."""
    import torch
    from scipy.stats import ks_2samp
    from paper_2605_16734_b200 import gcorbit as G
    st_o, t_o, s_o = _golden(config)
    f_o, lt_o = _loss(st_o, t_o)
    fld, spec, P, OF, GF, mu = make_case(config, N_ORACLE)
    if field == "hermite":
        GF.set_grid(101, 128, 128, kind=G.GC_GRID_HERMITE)
    s_n = np.arange(fld.ns) / (fld.ns - 1)
    chi = to_dev(fld.psi0 * (0.42 * s_n + 0.05 * s_n ** 2))     # iota = 0.42 + 0.1 s
    dt = 2e-8
    r = GF.trace_symplectic(spec.mass, spec.charge, to_dev(P.s), to_dev(P.theta), to_dev(P.zeta), to_dev(P.vpar),
                            to_dev(mu), chi, dt, int(round(T_MAX / dt)), s_loss=spec.s_loss, s_min=spec.s_min)
    torch.cuda.synchronize()
    st, t = r.status.cpu().numpy(), r.t.cpu().numpy()
    f_g, lt_g = _loss(st, t)
    se = 2.0 * np.sqrt(f_o * (1 - f_o) * 2.0 / N_ORACLE)
    p = ks_2samp(lt_g, lt_o).pvalue
    _record("symplectic_loss_statistics", config=config, field=field, dt=dt, oracle_loss_fraction=f_o,
            loss_fraction=f_g, bound=se, ks_p=float(p), status_equal=float((st == st_o).mean()),
            iterations_per_step=float(r.n_iter.sum().item()) / max(float(r.n_steps.sum().item()), 1.0))
    assert set(np.unique(st)) <= {0, 1, 2}
    assert (st == st_o).mean() >= 0.97, float((st == st_o).mean())   # paired: measured 98.5-98.9 %
    assert abs(f_g - f_o) <= se, (f_g, f_o, se)
    assert p > 0.01, p
