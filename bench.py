"""bench.py -- guiding-centre particle-steps/s (FP64) on B200, with roofline, end-to-end and CPU-oracle legs.

    python bench.py --gpus N --steps K --warmup W            # this repo's CUDA path (one rank per GPU)
    python bench.py --impl reference --gpus N --steps K --warmup W   # the CPU oracle, as it stands

Workload: BASELINE.json configs[3] -- the 1,000,000-particle trace north_star's target names: slowing-down alphas
with a (1-s)^2 birth profile in the static config-1 field (545 harmonics on 101 radial nodes), rtol = atol = 1e-8
(DESIGN.md section 7).  One "step" advances the whole ensemble by one segment of simulated time (default 2e-5 s,
about 350 Dormand-Prince attempts per particle) with ONE gc_trace call that continues the previous step in place
(GC_TRACE_RESUME), so K steps are the first (W + K) * segment seconds of the config-3 trace; lost particles drop
out as they do there.  A particle-step is one ATTEMPTED Dormand-Prince step (6 right-hand sides), accepted or
rejected.  --config 0|1|2|4 select the other BASELINE configurations (not the default line).

With --gpus N > 1 and no torchrun environment the script starts N ranks itself (torch.distributed.run on
127.0.0.1), one per GPU; every rank traces an independent draw of the same recipe (weak scaling, no data-path
collective).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "guiding-center particle-steps/s (FP64)"
UNIT = "particle-steps/s"
# FP64 ALU peak used as the roofline denominator: 148 SMs x 64 FP64 lanes x 2 flop
# x 1.965 GHz (sm_max_mhz in MEASURED_PEAKS.json) = 37.2 TFLOP/s; libgcprobes.so measures the sustained DFMA
# and DMMA rates of the same box in the same run, reported beside it.
FP64_LANES_PER_SM = 64


def flops_per_step(nh: int, M: int, nk: int, n_omega: int, per_harmonic: float = 28.0) -> float:
    """F_RHS = 28 nh + 18 (M + 1) + 350 (+ 75 K + 40 n_omega); F_step = 6 F_RHS + 250.
    per_harmonic = 28 is the survey's textbook count (14 FMA per harmonic); 16 is the cheapest exact formulation
    this build found (+-n pairing with slot-wise accumulation, 8 FMA per harmonic)."""
    f_rhs = per_harmonic * nh + 18.0 * (M + 1) + 350.0 + 75.0 * nk + 40.0 * n_omega
    return 6.0 * f_rhs + 250.0


DEFAULT_CONFIG = 3
FULL_SIZE = {0: 512, 1: 100_000, 2: 100_000, 3: 1_000_000, 4: 1_000_000}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference", "plumbing"],
                    help="cuda: this repo's kernels; reference: the CPU oracle; plumbing: launcher + process group + "
                         "timing reduction only (gloo, no device; used by the CPU tests)")
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG, choices=sorted(FULL_SIZE),
                    help="BASELINE.json config index (default 3: the 1M-particle trace)")
    ap.add_argument("--particles", type=int, default=None, help="particles per GPU (default: the config's)")
    ap.add_argument("--segment", type=float, default=2e-5, help="simulated seconds per step")
    ap.add_argument("--kernel", default="auto", choices=["auto", "mma", "tile", "warp", "generic"])
    ap.add_argument("--samples", type=int, default=0, help="NEXT-1: uniform-time samples per segment recorded by "
                    "gc_trace_sampled (0 = plain gc_trace, the default line); adds the P_zeta / weighted-Birkhoff "
                    "post-processing time to config")
    ap.add_argument("--slots", type=int, default=0, help="GC_OPT_WAVE_PARTICLES: record slots of the binned kernels "
                    "(0 = the library's default, 2^18)")
    ap.add_argument("--grid", default="", help="NEXT-2: NGSxNTHxNZE[:hermite] -- trace on the 3-D tricubic interpolant of B "
                    "(gc_field_set_grid) instead of the direct harmonic sum; not the default line")
    ap.add_argument("--symplectic", type=float, default=0.0, metavar="DT", help="NEXT-3: advance every segment with the "
                    "symplectic explicit-implicit Euler integrator at the fixed step DT seconds (gc_trace_symplectic) "
                    "instead of Dormand-Prince; a particle-step is then one symplectic step; static configs only; "
                    "not the default line")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t_start: float, t_end: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = [r for (ts, r) in self.rows if t_start <= ts <= t_end + 0.2 and len(r) >= 7] or \
               [r for (_, r) in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        num = lambda x: float(x) if x.replace(".", "", 1).isdigit() else float("nan")
        sm = sorted(num(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for j, nm in enumerate(names) if any(r[3 + j].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": num(rows[0][1]),
                "power_w_max": max(num(r[2]) for r in rows), "samples": len(rows), "reasons": reasons}


def workload(args, rank: int):
    from paper_2605_16734_b200 import workloads as W
    cfg = args.config
    fld, spec = W.make_field(cfg), W.make_spec(cfg)
    n = args.particles if args.particles else FULL_SIZE[cfg]
    P = W.make_particles(cfg, n, stream=rank)
    M = int(fld.xm.max())
    n_omega = len(set(np.asarray(fld.mode_omega).tolist()))
    info = {"workload": f"BASELINE.json configs[{cfg}]: {n} alphas per GPU, nh={fld.nh}, ns={fld.ns}, "
                        f"nk={fld.nk}, rtol={spec.rtol:g}, h_min={spec.h_min:g}; one step = one gc_trace call "
                        f"advancing the ensemble by {args.segment:g} s of simulated time (GC_TRACE_RESUME)",
            "particles_per_gpu": n, "segment_s": args.segment, "nh": fld.nh, "ns": fld.ns, "nk": fld.nk,
            "rtol": spec.rtol,
            "flop_per_particle_step": flops_per_step(fld.nh, M, fld.nk, n_omega),
            "flop_per_particle_step_min": flops_per_step(fld.nh, M, fld.nk, n_omega, per_harmonic=16.0)}
    return fld, spec, P, info


# ---- the CPU oracle legs -------------------------------------------------------------------------------------
def oracle_sample(fld, spec, P, seg: float, target_s: float):
    """Time the oracle, as it stands, on a bounded sample: the first n_s particles of the ensemble traced
    over [0, seg].  A pilot on 2 particles per thread sizes n_s for about target_s of wall time."""
    import oracle
    from paper_2605_16734_b200 import workloads as W
    OF = oracle.OracleField(fld)
    cores = oracle.num_threads()

    def run(k):
        Q = P.head(k)
        B = OF.eval_B_many(Q.s, Q.theta, Q.zeta)[:, 0]
        mu = W.mu_from(Q, B)
        t0 = time.perf_counter()
        r = OF.trace(spec, Q.s, Q.theta, Q.zeta, Q.vpar, mu, t0=0.0, t_max=seg)
        dt = time.perf_counter() - t0
        return int(r.n_acc.sum() + r.n_rej.sum()), dt

    k0 = min(P.n, 2 * cores)
    a0, d0 = run(k0)
    rate = a0 / max(d0, 1e-9)
    per_particle = a0 / k0
    k = int(min(P.n, max(k0, target_s * rate / max(per_particle, 1.0))))
    k = max(cores, (k // cores) * cores)
    a, d = run(k)
    return {"value": a / d, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {k} particles of the ensemble over [0, {seg:g}] s: {a} attempted steps in {d:.2f} s "
                      f"(oracle/gc_oracle.c, gcc -O2 -fopenmp, {cores} threads)"}


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step = one segment over a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    from paper_2605_16734_b200 import workloads as W
    fld, spec, P, info = workload(args, 0)
    OF = oracle.OracleField(fld)
    cores = oracle.num_threads()
    seg = args.segment
    # pilot: size the sample so that one step takes about cpu_seconds / (steps + warmup), at least one
    # particle per thread
    Q = P.head(min(P.n, 2 * cores))
    mu = W.mu_from(Q, OF.eval_B_many(Q.s, Q.theta, Q.zeta)[:, 0])
    t0 = time.perf_counter()
    r = OF.trace(spec, Q.s, Q.theta, Q.zeta, Q.vpar, mu, t0=0.0, t_max=seg)
    d0 = time.perf_counter() - t0
    per_step_budget = max(1.0, 4.0 * args.cpu_seconds / (args.steps + args.warmup))
    k = int(min(P.n, max(cores, Q.n * per_step_budget / max(d0, 1e-9))))
    k = min(P.n, max(cores, (k // cores) * cores))
    Q = P.head(k)
    mu = W.mu_from(Q, OF.eval_B_many(Q.s, Q.theta, Q.zeta)[:, 0])
    y = np.stack([Q.s, Q.theta, Q.zeta, Q.vpar])
    h = np.zeros(k)
    alive = np.arange(k)
    attempts, elapsed = 0, 0.0
    for step in range(args.warmup + args.steps):
        t_a, t_b = step * seg, (step + 1) * seg
        t0 = time.perf_counter()
        r = OF.trace(spec, y[0, alive], y[1, alive], y[2, alive], y[3, alive], mu[alive], h_in=h[alive],
                     t0=t_a, t_max=t_b)
        dt = time.perf_counter() - t0
        y[:, alive] = r.y
        h[alive] = r.h
        if step >= args.warmup:
            attempts += int(r.n_acc.sum() + r.n_rej.sum())
            elapsed += dt
        alive = alive[r.status == 0]
    value = attempts / elapsed
    sample = (f"first {k} particles of the ensemble, {args.steps} segments of {seg:g} s after {args.warmup} "
              f"warm-up segments: {attempts} attempted steps in {elapsed:.2f} s")
    info["particles_per_gpu"] = k
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * elapsed / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": info,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---- the CUDA arm ---------------------------------------------------------------------------------------------
def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2605_16734_b200 import build as B, ensemble as E, gcorbit as G, workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA arm has no CPU fallback (use --impl reference)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    if rank == 0:
        B.build()
    if world > 1:
        dist.barrier()

    fld, spec, P, info = workload(args, rank)
    n, seg, K, Wu = P.n, args.segment, args.steps, args.warmup
    GF = G.Field(fld)
    if args.kernel != "auto":
        GF.set_kernel({"warp": G.GC_KERNEL_WARP, "generic": G.GC_KERNEL_GENERIC, "tile": G.GC_KERNEL_TILE, "mma": G.GC_KERNEL_MMA}[args.kernel])
    if args.slots:
        GF.set_option(G.GC_OPT_WAVE_PARTICLES, args.slots)
    grid_kind = 0                                              # template argument of the lane kernels: 1 Lagrange, 2 Hermite
    if args.grid:
        gspec = args.grid.lower().split(":")
        grid_kind = 2 if len(gspec) > 1 and gspec[1].startswith("h") else 1
        GF.set_grid(*[int(x) for x in gspec[0].split("x")],
                    kind=G.GC_GRID_HERMITE if grid_kind == 2 else G.GC_GRID_LAGRANGE)
    kinfo = GF.kernel_info(n)
    kinfo["record_slots"] = args.slots if args.slots else "default"
    T = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
    s, th, ze, vpar = T(P.s), T(P.theta), T(P.zeta), T(P.vpar)
    Bst, _ = GF.field_eval(s, th, ze, derivs=False)          # mu = m v_perp^2 / (2 B) needs B at the start (A5)
    mu = T(0.5 * spec.mass * P.vperp2()) / Bst
    h = torch.zeros(n, dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)          # > 126 MB L2
    stream = torch.cuda.current_stream()

    def attempts_of(st):
        return int((st.n_acc.sum(dtype=torch.int64) + st.n_rej.sum(dtype=torch.int64)).item())

    def accepted_of(st):
        return int(st.n_acc.sum(dtype=torch.int64).item())

    # warm-up: the first W segments of the trace
    S = args.samples
    if args.symplectic > 0.0:
        s_n = np.arange(fld.ns) / (fld.ns - 1)
        chi = T(fld.psi0 * np.concatenate([[0.0], np.cumsum(0.5 * (fld.iota[1:] + fld.iota[:-1]) * np.diff(s_n))]))
        nst = max(1, int(round(seg / args.symplectic)))

        def resume(state, t0, t1):
            y = state.y
            return GF.trace_symplectic(spec.mass, spec.charge, y[0], y[1], y[2], y[3], mu, chi, args.symplectic, nst,
                                       t0=t0, out=state, flags=G.GC_TRACE_RESUME)
        state = GF.trace_symplectic(spec.mass, spec.charge, s, th, ze, vpar, mu, chi, args.symplectic, nst)
        state.n_acc, state.n_rej = state.n_steps, torch.zeros_like(state.n_steps)
        info["symplectic"] = {"dt": args.symplectic, "steps_per_segment": nst}
    elif S > 0:
        nsamp_total = S * (max(Wu, 1) + K) + 1
        sdt = seg / S

        def resume(state, t0, t1):
            y = state.y
            return GF.trace_sampled(spec, y[0], y[1], y[2], y[3], mu, 0.0, sdt, nsamp_total, h_inout=state.h, t0=t0,
                                    t_max=t1, out=state, flags=G.GC_TRACE_RESUME)
        state = GF.trace_sampled(spec, s, th, ze, vpar, mu, 0.0, sdt, nsamp_total, h_inout=h, t0=0.0, t_max=seg)
    else:
        def resume(state, t0, t1):
            return GF.trace_resume(spec, state, mu, t0=t0, t_max=t1)
        state = GF.trace(spec, s, th, ze, vpar, mu, h_inout=h, t0=0.0, t_max=seg)
    for w in range(1, max(Wu, 1)):
        resume(state, w * seg, (w + 1) * seg)
    torch.cuda.synchronize()
    first = max(Wu, 1)
    a_before = attempts_of(state)
    acc_before = accepted_of(state)
    alive_before = int((state.status == 0).sum().item())

    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local) if rank == 0 else None
    t_wall0 = time.time()
    for k in range(K):
        flush.fill_(k & 0xFF)                                  # L2 flush between timed iterations (not timed)
        ev[k][0].record(stream)
        resume(state, (first + k) * seg, (first + k + 1) * seg)
        ev[k][1].record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    step_ms = [a.elapsed_time(b) for a, b in ev]
    kernel_ms = float(sum(step_ms))
    attempts = attempts_of(state) - a_before
    accepted = accepted_of(state) - acc_before
    alive_after = int((state.status == 0).sum().item())
    ms_max, attempts_all = E.reduce_timing(kernel_ms, attempts, dev)
    value = attempts_all / (ms_max * 1e-3)

    # ---- NEXT-1 post-processing (only with --samples): P_zeta of every sample, weighted Birkhoff average per particle
    diag = None
    if S > 0:
        s_n = np.arange(fld.ns) / (fld.ns - 1)
        iota_int = np.concatenate([[0.0], np.cumsum(0.5 * (fld.iota[1:] + fld.iota[:-1]) * np.diff(s_n))])
        chi = T(fld.psi0 * iota_int)                                    # chi(s) = psi0 int iota ds (trapezoid on the nodes)
        tt = (torch.arange(nsamp_total, dtype=torch.float64, device=dev) * sdt).repeat_interleave(n)
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record(stream)
        pz = GF.pzeta_eval(spec.mass, spec.charge, state.samples.reshape(4, nsamp_total * n), tt, chi)
        e1.record(stream)
        wb = G.birkhoff(pz.reshape(nsamp_total, n), 0, state.sample_end)
        e2.record(stream)
        torch.cuda.synchronize()
        dig = wb[2][torch.isfinite(wb[2])]
        diag = {"samples_per_segment": S, "nsamp": nsamp_total, "sample_buffer_bytes": 32 * nsamp_total * n,
                "pzeta_eval_ms": e0.elapsed_time(e1), "birkhoff_ms": e1.elapsed_time(e2),
                "pzeta_points_per_s": nsamp_total * n / (e0.elapsed_time(e1) * 1e-3),
                "birkhoff_GBps": 8.0 * nsamp_total * n / (e1.elapsed_time(e2) * 1e-3) / 1e9,
                "digits_median": float(dig.median().item()) if dig.numel() else None,
                "frac_digits_below_3": float((dig < 3).double().mean().item()) if dig.numel() else None}

    # ---- e2e: the same segments through gc_trace_host, pinned host buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e and S == 0 and not args.symplectic:
        Ke = K                                                 # as many calls as timed steps: dilutes host-side stalls
        pin = lambda t: t.detach().cpu().pin_memory()
        hy, ht, hs, hh, hmu = pin(state.y), pin(state.t), pin(state.status), pin(state.h), pin(mu)
        hna, hnr, hnf = pin(state.n_acc), pin(state.n_rej), pin(state.n_forced)
        bufs = G.TraceResult(hy.numpy(), ht.numpy(), hs.numpy(), hna.numpy(), hnr.numpy(), hnf.numpy(), hh.numpy())
        yv = bufs.y
        a0 = int(bufs.n_acc.sum(dtype=np.int64) + bufs.n_rej.sum(dtype=np.int64))
        if world > 1:
            dist.barrier()
        # one untimed call first: it creates the field's host-path stream and device workspace
        GF.trace_host(spec, yv[0], yv[1], yv[2], yv[3], hmu.numpy(), t0=(first + K) * seg,
                      t_max=(first + K) * seg, bufs=bufs, flags=G.GC_TRACE_RESUME)
        t0 = time.perf_counter()
        per_call = []
        for k in range(Ke):
            tc = time.perf_counter()
            GF.trace_host(spec, yv[0], yv[1], yv[2], yv[3], hmu.numpy(), t0=(first + K + k) * seg,
                          t_max=(first + K + k + 1) * seg, bufs=bufs, flags=G.GC_TRACE_RESUME)
            per_call.append((time.perf_counter() - tc) * 1e3)
        dt_ms = (time.perf_counter() - t0) * 1e3
        a1 = int(bufs.n_acc.sum(dtype=np.int64) + bufs.n_rej.sum(dtype=np.int64))
        ms_e, att_e = E.reduce_timing(dt_ms, a1 - a0, dev)
        # bytes gc_trace_host copies per call under GC_TRACE_RESUME (gcorbit_api.cu): inputs 5 x 8n, h 8n,
        # y 32n, t 8n, status 4n, counters 12n in; y 32n, t 8n, status 4n, h 8n, counters 12n out
        e2e = {"value": att_e / (ms_e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 104 * n,
               "d2h_bytes_per_step": 64 * n, "steps": Ke, "ms_per_step": ms_e / Ke,
               "ms_per_call": [round(x, 2) for x in per_call],
               "ms_per_call_median": round(float(np.median(per_call)), 2),
               "api": "gc_trace_host (pinned host buffers; device workspace of the field reused between calls)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak_nominal = 148 * FP64_LANES_PER_SM * 2 * 1.965e9 / 1e12
    peak_src = "148 SMs x 64 FP64 lanes x 2 flop x 1965 MHz (fallback: MEASURED_PEAKS.json not found)"
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            mp = json.load(fh)
        sms = torch.cuda.get_device_properties(dev).multi_processor_count
        peak_nominal = sms * FP64_LANES_PER_SM * 2 * float(mp["sm_max_mhz"]) * 1e6 / 1e12
        peak_src = (f"{sms} SMs x 64 FP64 lanes x 2 flop x sm_max_mhz {mp['sm_max_mhz']:g} of MEASURED_PEAKS.json "
                    "(DESIGN.md section 6; the file holds no FP64 figure, so the ALU peak is derived)")
    except Exception:
        pass
    from bench_probes import probes
    probe_flops, _ = probes.dfma()
    dmma_flops, mixed_flops = probes.dmma()
    lds_distinct, lds_paired = probes.lds128()
    fstep, fstep_min = info["flop_per_particle_step"], info["flop_per_particle_step_min"]
    rate = attempts / (kernel_ms * 1e-3)                            # this rank's kernel, particle-steps/s
    achieved = rate * fstep / 1e12
    # constants of ncu --set full captures of the standard launches (profiles/ncu_constants.json.txt names each
    # capture): DRAM bytes per launch and executed FP64 flop per particle-step, per config.  They are used only when
    # the kernel sources are the ones that were profiled (hash stored beside them); any other workload or build: null.
    traffic = executed = cap_src = cap_stale = None
    std_launch = (args.particles is None and args.segment == 2e-5 and kinfo["kernel"] == "mma" and
                  args.samples == 0 and args.slots == 0 and not args.grid and not args.symplectic)
    tp = os.path.join(ROOT, "profiles", "ncu_constants.json.txt")
    if os.path.exists(tp) and std_launch:
        try:
            with open(tp) as fh:
                c = json.load(fh).get(f"config{args.config}", {})
            if c:
                cap_stale = c.get("kernel_source_hash") != kernel_source_hash()
                cap_src = c.get("source")
                if not cap_stale:
                    traffic, executed = c.get("dram_bytes_per_launch"), c.get("executed_flop_per_particle_step")
        except Exception:
            pass
    # frac / achieved: the FP64 flop the kernel really issues (ncu) where a capture of this build exists, else the
    # cheapest exact formulation (16 flop per harmonic); the survey's textbook count (28 flop per harmonic, work the
    # kernel does not do) is reported aside as frac_survey_model
    basis = "executed" if executed else "min_formulation"
    fbasis = executed if executed else fstep_min
    achieved_survey = achieved
    achieved = rate * fbasis / 1e12
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_nominal, "unit": "TFLOP/s",
                "frac": achieved / peak_nominal, "traffic": traffic, "frac_basis": basis,
                "flop_model": "frac / achieved count " + ("the FP64 flop the kernel issues (DMMA x 512 + DFMA x 2 + DMUL "
                              "+ DADD of the ncu capture named in ncu_capture)" if executed else "the cheapest exact "
                              "formulation (16 flop per harmonic and right-hand side; no ncu capture of this build and "
                              "workload)") + "; frac_survey_model counts the SURVEY.md 8(d) textbook formulation (28 flop "
                              "per harmonic), work this kernel does not do",
                "frac_survey_model": achieved_survey / peak_nominal,
                "frac_min_formulation": rate * fstep_min / 1e12 / peak_nominal,
                "frac_executed": (rate * executed / 1e12 / peak_nominal) if executed else None,
                "executed_flop_per_particle_step": executed, "ncu_capture": cap_src, "ncu_capture_stale": cap_stale,
                "kernel_source_hash": kernel_source_hash(),
                "kernel": f"trace_{kinfo['kernel']}_kernel", "launch_ms_avg": kernel_ms / K,
                "peak_source": peak_src,
                "peak_probe_tflops": probe_flops / 1e12, "peak_probe_dmma_tflops": dmma_flops / 1e12,
                "peak_probe_dmma_dfma_mixed_tflops": mixed_flops / 1e12,
                "lds128_cycles_per_warp_instr": {"distinct": lds_distinct, "lane_pairs_shared": lds_paired},
                "frac_of_probe": achieved / (probe_flops / 1e12),
                "flop_per_particle_step": fstep, "flop_per_particle_step_min": fstep_min,
                "particle_steps_per_launch": attempts / K}
    evals = 6.0                                                # Dormand-Prince: six new right-hand sides per attempt
    if args.symplectic > 0.0 or args.grid:
        # other formulations of the path (NEXT-2, NEXT-3): field evaluations per particle-step instead of the
        # Dormand-Prince count of 6
        if args.symplectic > 0.0:
            evals = float(state.n_iter.sum(dtype=torch.int64).item()) / max(attempts_of(state), 1)
            info["symplectic"]["field_evaluations_per_step"] = evals
        if args.grid:
            # gather-bound: 64 node values of 8 bytes per field evaluation come through the L1 data pipe from a table
            # that lives in L2; nominal pipe width 128 bytes per SM and cycle
            sms = torch.cuda.get_device_properties(dev).multi_processor_count
            gbytes = evals * 64.0 * 8.0
            peak_l1 = sms * 128.0 * peak_nominal * 1e12 / (sms * FP64_LANES_PER_SM * 2) / 1e9   # same clock as the ALU peak
            roofline = {"bound": "l1", "achieved": rate * gbytes / 1e9, "peak": peak_l1, "unit": "GB/s",
                        "frac": rate * gbytes / 1e9 / peak_l1, "traffic": None,
                        "model": f"{gbytes:.0f} gathered bytes per particle-step ({evals:.2f} evaluations of the "
                                 "tricubic interpolant x 64 nodes x 8 B) against sms x 128 B x 1.965 GHz of L1 data "
                                 "pipe; the table is read from L2, not HBM",
                        "fp64_frac": rate * (evals * 700.0 + 250.0) / 1e12 / peak_nominal,
                        "kernel": f"{'trace_symplectic_kernel' if args.symplectic > 0.0 else 'trace_lane_kernel'}<{grid_kind}>",
                        "launch_ms_avg": kernel_ms / K, "particle_steps_per_launch": attempts / K}
        else:
            # gc_trace_symplectic on the direct sum: the cell-binned mma engine from GC_TILE_MIN_PARTICLES(_SMALL) on
            # (unless GC_KERNEL_GENERIC is selected), else the lane kernel -- the rule of gcorbit_api.cu
            on_mma = kinfo["kernel"] == "mma"
            f_eval = ((fstep_min if on_mma else fstep) - 250.0) / 6.0
            roofline.update({"flop_per_particle_step": evals * f_eval, "achieved": rate * evals * f_eval / 1e12,
                             "frac": rate * evals * f_eval / 1e12 / peak_nominal, "frac_min_formulation": None,
                             "frac_executed": None, "frac_survey_model": None,
                             "frac_basis": "min_formulation" if on_mma else "survey_model",
                             "kernel": "trace_mma_symplectic_kernel" if on_mma else "trace_symplectic_kernel<0>",
                             "flop_model": ("cheapest exact count of one field evaluation (16 flop per harmonic) x "
                                            "measured evaluations per symplectic step, on the mma engine" if on_mma else
                                            "survey count of one field evaluation (28 flop per harmonic) x measured "
                                            "evaluations per symplectic step; the lane kernel evaluates the harmonic "
                                            "sum with one sincos per harmonic (generic engine)")})
    cpu = None
    if not args.no_cpu_baseline:
        cpu = oracle_sample(fld, spec, P, seg, args.cpu_seconds)
    if diag:
        info["next1_diagnostics"] = diag
    info.update({"kernel": kinfo, "l2": "flushed between timed steps (256 MiB write, outside each step's event pair)",
                 "alive_before": alive_before, "alive_after": alive_after,
                 "simulated_window_s": [first * seg, (first + K) * seg]})
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wu,
           "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "config": info,
           "rhs_evals_per_s": evals * value, "accepted_fraction": accepted / max(attempts, 1),
           "accepted_particle_steps_per_s": value * accepted / max(attempts, 1),
           "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": K, "clocks": clocks,
           "wall_s_timed_region": t_wall1 - t_wall0}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def kernel_source_hash() -> str:
    """Hash of the sources trace_mma_kernel is compiled from; stored beside the ncu constants of
    profiles/ncu_constants.json.txt so that a later build does not quote an earlier build's counters."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_2605_16734_b200", "csrc")
    for name in ("device_math.cuh", "field.cuh", "kernels_generic.cuh", "kernels_tile.cuh", "kernels_mma.cuh"):
        with open(os.path.join(csrc, name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def run_plumbing(args):
    """--impl plumbing: everything of the multi-rank path that is not a kernel -- launch, rendezvous, process group
    (gloo, CPU), the max-over-ranks / sum-over-ranks reduction of ensemble.reduce_timing and the rank-0 JSON line --
    with made-up per-rank numbers.  Used by tests/test_bench_contract.py; measures nothing."""
    import torch.distributed as dist
    from paper_2605_16734_b200 import ensemble as E
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
    ms, attempts = E.reduce_timing(100.0 + rank, 1000 * (rank + 1))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"impl": "plumbing", "n_gpus": world, "ms_max": ms, "attempts_sum": attempts}))


def launch_ranks(args) -> int:
    """`python bench.py --gpus N` without a torchrun environment: start N ranks of this script on this node
    (torch.distributed.run, rendezvous on 127.0.0.1, a free port), one per GPU, and pass their output through."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")                      # communicator / rank lines (WARN prints none)
    env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    return subprocess.call(cmd, env=env)


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(launch_ranks(args))
    if args.impl == "reference":
        run_reference(args)
    elif args.impl == "plumbing":
        run_plumbing(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
