"""Writes tests/golden/statistics_config{1,2,3,4}.txt: ORACLE ensembles for the loss-fraction / loss-time acceptance
of BASELINE.json north_star ("Ensemble loss fractions must agree within the Monte Carlo standard error, with
loss-time histograms passing a two-sample KS test at p>0.01 ... on all five configs"; the paper's own comparison of
two codes: PAPER.md:68,72, 5000 particles, identical loss fractions).

Calls ONLY oracle/ and the seeded input recipes (paper_2605_16734_b200/workloads.py); nothing of the CUDA path.

    python tests/golden/make_statistics_golden.py [--configs 1 2 3 4] [--particles 2048] [--t-max 1e-3]

Size as SURVEY.md section 8(d) asks: 2048 particles per config traced to 1e-3 s (150-400 loss events each), about
5-10 minutes per config on 16 host threads.  Ensemble: workloads.make_particles(config, 2048) (its own seeded draw
of that size), mu from the oracle's B at the start point; config 1 keeps its h_min = 1e-12.  Config 0 (512 particles
on s = 0.25, 1e-4 s; the oracle loses 40 of them inside that horizon) is too small for statistics and is
compared particle by particle, status included, instead (tests/test_gpu_parity.py).  Columns: status, t_out [s], s_out, attempted steps.
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--configs", type=int, nargs="+", default=[1, 2, 3, 4])
    ap.add_argument("--particles", type=int, default=2048)
    ap.add_argument("--t-max", type=float, default=1e-3)
    ap.add_argument("--out-dir", default=HERE)
    args = ap.parse_args()
    import oracle
    from paper_2605_16734_b200 import workloads as W
    for cfg in args.configs:
        fld, spec = W.make_field(cfg), W.make_spec(cfg)
        P = W.make_particles(cfg, args.particles)
        OF = oracle.OracleField(fld)
        mu = W.mu_from(P, OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
        t0 = time.time()
        r = OF.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=args.t_max)
        dt = time.time() - t0
        attempts = r.n_acc.astype(np.int64) + r.n_rej
        head = (f"oracle ensemble, BASELINE.json configs[{cfg}]: workloads.make_particles({cfg}, {args.particles}), "
                f"t_max = {args.t_max:g} s, rtol = {spec.rtol:g}, h_min = {spec.h_min:g}\n"
                f"written by: python tests/golden/make_statistics_golden.py --configs {cfg} --particles "
                f"{args.particles} --t-max {args.t_max:g}   ({oracle.num_threads()} threads, {dt:.0f} s, "
                f"{int(attempts.sum())} attempted steps)\n"
                f"lost {int((r.status == 1).sum())}, axis {int((r.status == 2).sum())}, "
                f"at t_max {int((r.status == 0).sum())}, other {int((r.status > 2).sum())}\n"
                "status t_out s_out attempts")
        out = os.path.join(args.out_dir, f"statistics_config{cfg}.txt")
        np.savetxt(out, np.column_stack([r.status, r.t, r.y[0], attempts]), fmt=["%d", "%.17g", "%.17g", "%d"],
                   header=head)
        print(f"config {cfg}: {dt:.0f} s, lost {(r.status == 1).mean():.4f}, axis {(r.status == 2).mean():.4f} -> {out}",
              flush=True)


if __name__ == "__main__":
    main()
