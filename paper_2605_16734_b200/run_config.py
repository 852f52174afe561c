"""Trace one of the BASELINE.json configurations to its full horizon on one GPU and print the job's results as JSON:
loss fraction versus time, status counts, attempted steps, device time, energy conservation of the survivors
(static fields) and, for config 4, the number of Poincare records.

    python -m paper_2605_16734_b200.run_config --config 1 [--segments 100] [--particles N] [--t-max T]
                                               [--grid NGSxNTHxNZE[:hermite]]     (NEXT-2: trace on the interpolant)

The horizon is cut into equal segments traced in place with GC_TRACE_RESUME (A24: the last step of each
segment is clipped to the segment end).  Everything runs in the CUDA kernels behind the C ABI; there is no CPU path.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--segments", type=int, default=100)
    ap.add_argument("--particles", type=int, default=None)
    ap.add_argument("--t-max", type=float, default=None, help="horizon in seconds (default: the config's)")
    ap.add_argument("--poincare-per-particle", type=int, default=8, help="config 4: record capacity per particle")
    ap.add_argument("--grid", default="", help="NGSxNTHxNZE[:hermite]: trace on the 3-D tricubic interpolant of B; mu and the "
                    "energy check still use the direct sum at the start and end points")
    args = ap.parse_args()

    import torch
    from . import gcorbit as G, workloads as W

    dev = torch.device("cuda:0")
    fld, spec = W.make_field(args.config), W.make_spec(args.config)
    P = W.make_particles(args.config, args.particles)
    n = P.n
    t_max = args.t_max if args.t_max else spec.t_max
    seg = t_max / args.segments
    GF = G.Field(fld)
    T = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
    s, th, ze, vpar = T(P.s), T(P.theta), T(P.zeta), T(P.vpar)
    B0, _ = GF.field_eval(s, th, ze, derivs=False)
    mu = T(0.5 * spec.mass * P.vperp2()) / B0
    E0 = 0.5 * spec.mass * vpar ** 2 + mu * B0
    if args.grid:
        gspec = args.grid.lower().split(":")
        GF.set_grid(*[int(x) for x in gspec[0].split("x")],
                    kind=G.GC_GRID_HERMITE if len(gspec) > 1 and gspec[1].startswith("h") else G.GC_GRID_LAGRANGE)
    h = torch.zeros(n, dtype=torch.float64, device=dev)
    cap = args.poincare_per_particle * n if args.config == 4 else 0
    stream = torch.cuda.current_stream()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    records = 0
    device_ms = 0.0
    curve = []
    wall0 = time.time()
    state = None
    for k in range(args.segments):
        t0, t1 = k * seg, (t_max if k == args.segments - 1 else (k + 1) * seg)
        ev0.record(stream)
        if state is None:
            state = GF.trace(spec, s, th, ze, vpar, mu, h_inout=h, t0=t0, t_max=t1, poincare_capacity=cap)
        else:
            state = GF.trace_resume(spec, state, mu, t0=t0, t_max=t1, poincare_capacity=cap)
        ev1.record(stream)
        torch.cuda.synchronize()
        device_ms += ev0.elapsed_time(ev1)
        if cap:
            G.finish_poincare(state)
            records += state.poincare_count
            state.poincare = torch.empty((cap, 4), dtype=torch.float64, device=dev)
        st = state.status
        curve.append({"t": t1, "lost": float((st == G.ST_LOST).double().mean().item()),
                      "running": int((st == G.ST_TMAX).sum().item())})
    wall = time.time() - wall0

    st = state.status.cpu().numpy()
    attempts = int(state.n_acc.sum(dtype=torch.int64).item() + state.n_rej.sum(dtype=torch.int64).item())
    out = {"config": args.config, "particles": n, "t_max": t_max, "segments": args.segments, "grid": args.grid or None,
           "kernel": GF.kernel_info(n), "attempted_steps": attempts,
           "accepted_fraction": float(state.n_acc.sum(dtype=torch.int64).item()) / max(attempts, 1),
           "forced_min_steps": int(state.n_forced.sum(dtype=torch.int64).item()),
           "device_s": device_ms * 1e-3, "wall_s": wall, "particle_steps_per_s": attempts / (device_ms * 1e-3),
           "status_counts": {name: int((st == code).sum()) for name, code in
                             (("t_max", 0), ("lost", 1), ("axis", 2), ("max_steps", 3), ("non_finite", 4))},
           "loss_fraction": float((st == 1).mean())}
    lost_t = state.t.cpu().numpy()[st == 1]
    if lost_t.size:
        edges = np.logspace(np.log10(max(lost_t.min(), 1e-7)), np.log10(t_max), 13)
        hist, _ = np.histogram(lost_t, bins=edges)
        out["loss_time_histogram"] = {"edges_s": [float(f"{e:.3e}") for e in edges], "counts": hist.tolist()}
        out["first_loss_s"] = float(lost_t.min())
    pick = [c for i, c in enumerate(curve) if (i + 1) % max(1, args.segments // 20) == 0 or i == len(curve) - 1]
    out["loss_fraction_vs_time"] = [{"t": float(f"{c['t']:.4e}"), "lost": round(c["lost"], 6)} for c in pick]
    if fld.nk == 0:                                            # static field: energy of the survivors is conserved
        surv = state.status == G.ST_TMAX
        y = state.y
        if args.grid:
            GF.set_grid(0, 0, 0)                               # energy with the direct sum at both ends
        B1, _ = GF.field_eval(y[0].contiguous(), y[1].contiguous(), y[2].contiguous(), derivs=False)
        E1 = 0.5 * spec.mass * y[3] ** 2 + mu * B1
        rel = ((E1 - E0) / E0).abs()[surv]
        if rel.numel():
            out["energy_drift_survivors"] = {"median": float(rel.median().item()), "max": float(rel.max().item())}
    if cap:
        out["poincare_records"] = records
    print(json.dumps(out))


if __name__ == "__main__":
    main()
