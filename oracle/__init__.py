"""CPU ORACLE bindings -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see gc_oracle.h).

ctypes wrapper around ``oracle/libgc_oracle.so`` (plain C, built by :func:`build`).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import
this package.  It shares nothing with ``paper_2605_16734_b200/csrc``.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libgc_oracle.so")
_SRC = os.path.join(_HERE, "gc_oracle.c")
_HDR = os.path.join(_HERE, "gc_oracle.h")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp, no fast-math, no FMA contraction."""
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return _SO
    cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-ffp-contract=off",
           "-Wall", "-Wextra", _SRC, "-o", _SO, "-lm"]
    subprocess.run(cmd, check=True)
    return _SO


class _Desc(C.Structure):
    _fields_ = [("ns", C.c_int32), ("nfp", C.c_int32), ("nh", C.c_int32),
                ("xm", C.c_void_p), ("xn", C.c_void_p), ("bmnc", C.c_void_p),
                ("G", C.c_void_p), ("I", C.c_void_p), ("iota", C.c_void_p),
                ("psi0", C.c_double), ("nk", C.c_int32),
                ("mode_m", C.c_void_p), ("mode_n", C.c_void_p),
                ("mode_omega", C.c_void_p), ("mode_phase", C.c_void_p), ("phihat", C.c_void_p),
                ("bmns", C.c_void_p), ("kmnc", C.c_void_p), ("kmns", C.c_void_p)]


class _Params(C.Structure):
    _fields_ = [("mass", C.c_double), ("charge", C.c_double), ("t0", C.c_double), ("t_max", C.c_double),
                ("rtol", C.c_double), ("atol", C.c_double), ("v_ref", C.c_double),
                ("h0", C.c_double), ("h_min", C.c_double), ("s_loss", C.c_double), ("s_min", C.c_double),
                ("max_steps", C.c_int64), ("poincare_capacity", C.c_int64), ("traj_capacity", C.c_int64),
                ("section", C.c_int64), ("refine_loss", C.c_int64)]


class _SymParams(C.Structure):
    _fields_ = [("mass", C.c_double), ("charge", C.c_double), ("t0", C.c_double), ("dt", C.c_double),
                ("nsteps", C.c_int64), ("s_loss", C.c_double), ("s_min", C.c_double), ("newton_tol", C.c_double)]


def _load():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.oracle_field_create.restype = C.c_void_p
        L.oracle_field_create.argtypes = [C.POINTER(_Desc)]
        L.oracle_field_destroy.argtypes = [C.c_void_p]
        L.oracle_scale_accept.restype = C.c_double
        L.oracle_scale_accept.argtypes = [C.c_double]
        L.oracle_scale_reject.restype = C.c_double
        L.oracle_scale_reject.argtypes = [C.c_double]
        L.oracle_err_norm.restype = C.c_double
        L.oracle_num_threads.restype = C.c_int
        L.oracle_trace.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def lagrange(ns: int, s: float):
    i0 = C.c_int32(0)
    w = np.zeros(4)
    dw = np.zeros(4)
    _load().oracle_lagrange(C.c_int32(ns), C.c_double(s), C.byref(i0), _p(w), _p(dw))
    return int(i0.value), w, dw


def scale_accept(err: float) -> float:
    return float(_load().oracle_scale_accept(err))


def scale_reject(err: float) -> float:
    return float(_load().oracle_scale_reject(err))


def err_norm(y, y_new, delta, rtol, atol) -> float:
    y, y_new, delta = _f64(y), _f64(y_new), _f64(delta)
    return float(_load().oracle_err_norm(_p(y), _p(y_new), _p(delta), C.c_double(rtol), C.c_double(atol)))


def dp5_dense(y, y_new, k, h, tau):
    y, y_new, k = _f64(y), _f64(y_new), _f64(k)
    assert k.shape == (7, 4)
    out = np.zeros(4)
    _load().oracle_dp5_dense(_p(y), _p(y_new), _p(k), C.c_double(h), C.c_double(tau), _p(out))
    return out


@dataclass
class TraceResult:
    y: np.ndarray          # [4][n]: s, theta, zeta, v_par (m/s)
    t: np.ndarray          # [n]
    status: np.ndarray     # [n] int32
    n_acc: np.ndarray
    n_rej: np.ndarray
    n_forced: np.ndarray
    h: np.ndarray          # [n] next step proposal
    poincare: np.ndarray | None = None      # [count][4]
    poincare_count: int = 0
    traj: np.ndarray | None = None          # [n][cap][5]
    traj_count: np.ndarray | None = None


@dataclass
class SymplecticResult:
    y: np.ndarray          # [4][n]: s, theta, zeta, v_par (m/s)
    t: np.ndarray          # [n]
    status: np.ndarray     # [n] int32: 0 all steps done, 1 lost, 2 axis, 4 Newton failure / non-finite
    n_steps: np.ndarray
    n_iter: np.ndarray
    samples: np.ndarray | None = None       # [4][nsamp][n]
    sample_end: np.ndarray | None = None


class OracleField:
    """Host tables copied into the C oracle (oracle_field_create)."""

    def __init__(self, fld):
        L = _load()
        self._keep = dict(
            xm=_i32(fld.xm), xn=_i32(fld.xn), bmnc=_f64(fld.bmnc), G=_f64(fld.G), I=_f64(fld.I),
            iota=_f64(fld.iota), mode_m=_i32(fld.mode_m), mode_n=_i32(fld.mode_n),
            mode_omega=_f64(fld.mode_omega), mode_phase=_f64(fld.mode_phase), phihat=_f64(fld.phihat))
        k = self._keep
        for name in ("bmns", "kmnc", "kmns"):                      # NEXT-4 tables: absent = None
            a = getattr(fld, name, None)
            k[name] = None if a is None else _f64(a)
        self.ns, self.nh, self.nk = int(fld.ns), int(k["xm"].shape[0]), int(k["mode_m"].shape[0])
        assert k["bmnc"].shape == (self.ns, self.nh)
        assert all(k[nm] is None or k[nm].shape == (self.ns, self.nh) for nm in ("bmns", "kmnc", "kmns"))
        if self.nk:
            assert k["phihat"].shape == (self.ns, self.nk)
        d = _Desc(self.ns, int(fld.nfp), self.nh, _p(k["xm"]), _p(k["xn"]), _p(k["bmnc"]),
                  _p(k["G"]), _p(k["I"]), _p(k["iota"]), float(fld.psi0), self.nk,
                  _p(k["mode_m"]), _p(k["mode_n"]), _p(k["mode_omega"]), _p(k["mode_phase"]),
                  _p(k["phihat"]), _p(k["bmns"]), _p(k["kmnc"]), _p(k["kmns"]))
        self._h = C.c_void_p(L.oracle_field_create(C.byref(d)))
        if not self._h.value:
            raise ValueError("oracle_field_create rejected the description")
        self.psi0 = float(fld.psi0)

    def __del__(self):
        try:
            if self._h.value:
                _load().oracle_field_destroy(self._h)
                self._h = C.c_void_p(None)
        except Exception:
            pass

    # ---- point evaluations ---------------------------------------------------------------------------
    def eval_B(self, s, th, ze):
        out = np.zeros(4)
        _load().oracle_eval_B(self._h, C.c_double(s), C.c_double(th), C.c_double(ze), _p(out))
        return out

    def eval_B_many(self, s, th, ze):
        s, th, ze = np.broadcast_arrays(_f64(s), _f64(th), _f64(ze))
        out = np.zeros((s.size, 4))
        for i, (a, b, c) in enumerate(zip(s.ravel(), th.ravel(), ze.ravel())):
            out[i] = self.eval_B(a, b, c)
        return out

    # ---- NEXT-2: local tricubic interpolant of B on an (s, theta, zeta) grid ----------------------------
    def set_grid(self, ngs: int, nth: int, nze: int):
        """Tabulate B by the direct sum and evaluate it from now on as a tensor-product cubic Lagrange
        interpolant (reading A27); (0, 0, 0) switches back to the direct sum."""
        if _load().oracle_field_set_grid(self._h, C.c_int32(ngs), C.c_int32(nth), C.c_int32(nze)) != 0:
            raise ValueError("oracle_field_set_grid: each grid size must be >= 4 (or all 0)")
        self.grid_shape = (ngs, nth, nze) if ngs else None

    def grid(self) -> np.ndarray:
        L = _load()
        L.oracle_field_grid.restype = C.POINTER(C.c_double)
        L.oracle_field_grid.argtypes = [C.c_void_p]
        ptr = L.oracle_field_grid(self._h)
        return np.ctypeslib.as_array(ptr, shape=self.grid_shape).copy()

    def set_grid_hermite(self, ngs: int, nth: int, nze: int):
        """Second reading of NEXT-2 (A31): the C1 tricubic Hermite interpolant on the same node grid."""
        if _load().oracle_field_set_grid_hermite(self._h, C.c_int32(ngs), C.c_int32(nth), C.c_int32(nze)) != 0:
            raise ValueError("oracle_field_set_grid_hermite: each grid size must be >= 2 (or all 0)")
        self.grid_shape = (ngs, nth, nze) if ngs else None

    def grid8(self) -> np.ndarray:
        L = _load()
        L.oracle_field_grid8.restype = C.POINTER(C.c_double)
        L.oracle_field_grid8.argtypes = [C.c_void_p]
        ptr = L.oracle_field_grid8(self._h)
        return np.ctypeslib.as_array(ptr, shape=self.grid_shape + (8,)).copy()

    def eval_B_mixed(self, s, th, ze):
        out = np.zeros(8)
        _load().oracle_eval_B_mixed(self._h, C.c_double(s), C.c_double(th), C.c_double(ze), _p(out))
        return out

    def eval_B_sum(self, s, th, ze):
        out = np.zeros(4)
        _load().oracle_eval_B_sum(self._h, C.c_double(s), C.c_double(th), C.c_double(ze), _p(out))
        return out

    def eval_K(self, s, th, ze):
        out = np.zeros(4)
        _load().oracle_eval_K(self._h, C.c_double(s), C.c_double(th), C.c_double(ze), _p(out))
        return out

    def rhs_general(self, mass, charge, mu, v_ref, t, y):
        y = _f64(y)
        out = np.zeros(4)
        _load().oracle_rhs_general(self._h, C.c_double(mass), C.c_double(charge), C.c_double(mu),
                                   C.c_double(v_ref), C.c_double(t), _p(y), _p(out))
        return out

    def eval_profiles(self, s):
        out = np.zeros(6)
        _load().oracle_eval_profiles(self._h, C.c_double(s), _p(out))
        return out

    def eval_pert(self, s, th, ze, t):
        out = np.zeros(9)
        _load().oracle_eval_pert(self._h, C.c_double(s), C.c_double(th), C.c_double(ze), C.c_double(t),
                                 _p(out))
        return out

    def rhs(self, mass, charge, mu, v_ref, t, y):
        y = _f64(y)
        out = np.zeros(4)
        _load().oracle_rhs(self._h, C.c_double(mass), C.c_double(charge), C.c_double(mu),
                           C.c_double(v_ref), C.c_double(t), _p(y), _p(out))
        return out

    def dp5_attempt(self, mass, charge, mu, v_ref, t, y, k1, h):
        y, k1 = _f64(y), _f64(k1)
        y_new, k, delta = np.zeros(4), np.zeros((7, 4)), np.zeros(4)
        _load().oracle_dp5_attempt(self._h, C.c_double(mass), C.c_double(charge), C.c_double(mu),
                                   C.c_double(v_ref), C.c_double(t), _p(y), _p(k1), C.c_double(h),
                                   _p(y_new), _p(k), _p(delta))
        return y_new, k, delta

    # ---- ensembles -----------------------------------------------------------------------------------
    def trace(self, spec, s0, th0, ze0, vpar0, mu, h_in=None, poincare_capacity=0, traj_capacity=0,
              t0=None, t_max=None, section=0, refine_loss=False) -> TraceResult:
        s0, th0, ze0, vpar0, mu = map(_f64, (s0, th0, ze0, vpar0, mu))
        n = s0.shape[0]
        p = _Params(spec.mass, spec.charge, spec.t0 if t0 is None else t0,
                    spec.t_max if t_max is None else t_max, spec.rtol, spec.atol, spec.v_ref,
                    spec.h0, spec.h_min, spec.s_loss, spec.s_min, int(spec.max_steps),
                    int(poincare_capacity), int(traj_capacity), int(section), int(bool(refine_loss)))
        h = np.zeros(n) if h_in is None else _f64(h_in).copy()
        y = np.zeros((4, n))
        t = np.zeros(n)
        status = np.zeros(n, np.int32)
        n_acc, n_rej, n_forced = (np.zeros(n, np.int32) for _ in range(3))
        pc = np.zeros((max(poincare_capacity, 1), 4)) if poincare_capacity else None
        pcount = C.c_int64(0)
        traj = np.zeros((n, traj_capacity, 5)) if traj_capacity else None
        tcount = np.zeros(n, np.int64) if traj_capacity else None
        rc = _load().oracle_trace(self._h, C.byref(p), C.c_int64(n), _p(s0), _p(th0), _p(ze0), _p(vpar0),
                                  _p(mu), _p(h), _p(y), _p(t), _p(status), _p(n_acc), _p(n_rej),
                                  _p(n_forced), _p(pc), C.byref(pcount) if poincare_capacity else None,
                                  _p(traj), _p(tcount))
        if rc != 0:
            raise ValueError("oracle_trace: bad arguments")
        res = TraceResult(y, t, status, n_acc, n_rej, n_forced, h)
        if poincare_capacity:
            res.poincare_count = int(pcount.value)
            res.poincare = pc[:min(res.poincare_count, poincare_capacity)]
        if traj_capacity:
            res.traj, res.traj_count = traj, tcount
        return res

    def trace_sampled(self, spec, s0, th0, ze0, vpar0, mu, sample_t0, sample_dt, nsamp, h_in=None, t0=None,
                      t_max=None) -> TraceResult:
        """O9: the trace with uniform-time samples of the continuous extension; adds ``samples`` [4][nsamp][n]
        and ``nsampled`` [n] (= sample_end: one past the last sample index written) to the result."""
        s0, th0, ze0, vpar0, mu = map(_f64, (s0, th0, ze0, vpar0, mu))
        n = s0.shape[0]
        p = _Params(spec.mass, spec.charge, spec.t0 if t0 is None else t0,
                    spec.t_max if t_max is None else t_max, spec.rtol, spec.atol, spec.v_ref,
                    spec.h0, spec.h_min, spec.s_loss, spec.s_min, int(spec.max_steps), 0, 0)
        h = np.zeros(n) if h_in is None else _f64(h_in).copy()
        y = np.zeros((4, n))
        t = np.zeros(n)
        status = np.zeros(n, np.int32)
        n_acc, n_rej, n_forced = (np.zeros(n, np.int32) for _ in range(3))
        samples = np.full((4, int(nsamp), n), np.nan)
        nsampled = np.zeros(n, np.int32)
        L = _load()
        L.oracle_trace_sampled.argtypes = [C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 12 + \
            [C.c_double, C.c_double, C.c_int64, C.c_void_p, C.c_void_p]
        rc = L.oracle_trace_sampled(self._h, C.byref(p), C.c_int64(n), _p(s0), _p(th0), _p(ze0), _p(vpar0),
                                    _p(mu), _p(h), _p(y), _p(t), _p(status), _p(n_acc), _p(n_rej), _p(n_forced),
                                    float(sample_t0), float(sample_dt), int(nsamp), _p(samples), _p(nsampled))
        if rc != 0:
            raise ValueError("oracle_trace_sampled: bad arguments")
        res = TraceResult(y, t, status, n_acc, n_rej, n_forced, h)
        res.samples, res.nsampled = samples, nsampled
        return res

    def pzeta(self, mass, charge, chi_nodes, s, th, ze, vpar, t):
        """A17: P_zeta at arrays of states and times (broadcast)."""
        chi_nodes = _f64(chi_nodes)
        L = _load()
        L.oracle_pzeta.restype = C.c_double
        L.oracle_pzeta.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p] + [C.c_double] * 5
        s, th, ze, vpar, t = np.broadcast_arrays(*(np.asarray(a, float) for a in (s, th, ze, vpar, t)))
        out = np.empty(s.shape)
        for idx in np.ndindex(s.shape):
            out[idx] = L.oracle_pzeta(self._h, mass, charge, _p(chi_nodes), s[idx], th[idx], ze[idx], vpar[idx], t[idx])
        return out

    # ---- NEXT-3: symplectic explicit-implicit Euler (static fields, K = 0) ---------------------------------------
    def symplectic_step(self, mass, charge, mu, chi_nodes, h, z, newton_tol=1e-13):
        """One step on z = (s, theta, zeta, p_zeta); returns (z_new, Newton iterations)."""
        chi_nodes, z = _f64(chi_nodes), _f64(z).copy()
        it = C.c_int32(0)
        L = _load()
        L.oracle_symplectic_step.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_double,
                                             C.c_double, C.c_void_p, C.c_void_p]
        rc = L.oracle_symplectic_step(self._h, mass, charge, mu, _p(chi_nodes), h, newton_tol, _p(z), C.byref(it))
        if rc != 0:
            raise ArithmeticError("oracle_symplectic_step: Newton did not converge")
        return z, int(it.value)

    def symplectic_pzeta(self, mass, charge, chi_nodes, s, th, ze, vpar):
        chi_nodes = _f64(chi_nodes)
        L = _load()
        L.oracle_symplectic_pzeta.restype = C.c_double
        L.oracle_symplectic_pzeta.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p] + [C.c_double] * 4
        return L.oracle_symplectic_pzeta(self._h, mass, charge, _p(chi_nodes), s, th, ze, vpar)

    def symplectic_vpar(self, mass, charge, chi_nodes, s, th, ze, pz):
        chi_nodes = _f64(chi_nodes)
        L = _load()
        L.oracle_symplectic_vpar.restype = C.c_double
        L.oracle_symplectic_vpar.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p] + [C.c_double] * 4
        return L.oracle_symplectic_vpar(self._h, mass, charge, _p(chi_nodes), s, th, ze, pz)

    def trace_symplectic(self, mass, charge, s0, th0, ze0, vpar0, mu, chi_nodes, dt, nsteps, t0=0.0, s_loss=1.0,
                         s_min=1e-3, newton_tol=1e-13, sample_stride=0, nsamp=0):
        """n particles, nsteps fixed steps each; returns a SymplecticResult."""
        s0, th0, ze0, vpar0, mu, chi_nodes = map(_f64, (s0, th0, ze0, vpar0, mu, chi_nodes))
        n = s0.shape[0]
        p = _SymParams(mass, charge, t0, dt, int(nsteps), s_loss, s_min, newton_tol)
        y, t = np.zeros((4, n)), np.zeros(n)
        status, steps, iters = (np.zeros(n, np.int32) for _ in range(3))
        samples = np.full((4, int(nsamp), n), np.nan) if nsamp else None
        send = np.zeros(n, np.int32) if nsamp else None
        L = _load()
        L.oracle_trace_symplectic.argtypes = [C.c_void_p, C.c_void_p, C.c_int64] + [C.c_void_p] * 11 + \
            [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
        rc = L.oracle_trace_symplectic(self._h, C.byref(p), n, _p(s0), _p(th0), _p(ze0), _p(vpar0), _p(mu),
                                       _p(chi_nodes), _p(y), _p(t), _p(status), _p(steps), _p(iters),
                                       int(sample_stride), int(nsamp), _p(samples), _p(send))
        if rc != 0:
            raise ValueError("oracle_trace_symplectic: bad arguments")
        return SymplecticResult(y, t, status, steps, iters, samples, send)

    def rk4(self, mass, charge, v_ref, s0, th0, ze0, vpar0, mu, t0, h, nsteps):
        s0, th0, ze0, vpar0, mu = map(_f64, (s0, th0, ze0, vpar0, mu))
        n = s0.shape[0]
        y = np.zeros((4, n))
        _load().oracle_rk4(self._h, C.c_double(mass), C.c_double(charge), C.c_double(v_ref), C.c_int64(n),
                           _p(s0), _p(th0), _p(ze0), _p(vpar0), _p(mu), C.c_double(t0), C.c_double(h),
                           C.c_int64(nsteps), _p(y))
        return y


_RHS_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double))


def dp5_attempt_fn(fun, t, y, h, k1=None):
    """One Dormand-Prince attempt on an arbitrary Python right-hand side ``fun(t, y[4]) -> dydt[4]``
    (tableau pins only)."""
    y = _f64(y)

    def _cb(_ctx, tt, yp, dp):
        out = fun(tt, np.array([yp[i] for i in range(4)]))
        for i in range(4):
            dp[i] = float(out[i])

    cb = _RHS_FN(_cb)
    k1 = _f64(fun(t, y.copy())) if k1 is None else _f64(k1)
    y_new, k, delta = np.zeros(4), np.zeros((7, 4)), np.zeros(4)
    _load().oracle_dp5_attempt_fn(cb, None, C.c_double(t), _p(y), _p(k1), C.c_double(h),
                                  _p(y_new), _p(k), _p(delta))
    return y_new, k, delta


# ---- weighted Birkhoff average (NEXT-1; PAPER.md:50,94 cite Duignan & Meiss 2023) -----------------------------
def birkhoff_weights(N: int) -> np.ndarray:
    """w_j = g((j + 1) / (N + 1)), g(x) = exp(-1 / (x (1 - x))), j = 0 .. N-1: the C-infinity bump of the weighted
    Birkhoff average, sampled strictly inside (0, 1) so that no weight is 0/0."""
    x = (np.arange(N) + 1.0) / (N + 1.0)
    return np.exp(-1.0 / (x * (1.0 - x)))


def birkhoff_average(f) -> float:
    """WB_N(f) = sum_j w_j f_j / sum_j w_j."""
    f = np.asarray(f, float)
    w = birkhoff_weights(f.shape[0])
    return float(np.sum(w * f) / np.sum(w))


def birkhoff_digits(f):
    """(WB of the first half, WB of the second half, digit accuracy): the series is cut into two halves of
    N = len(f) // 2 samples; digits = -log10(|WB_1 - WB_2| / max(|WB_1|, |WB_2|)), capped at 16 (reading A25 of
    DESIGN.md: an orbit on an invariant torus gives many digits, a chaotic one few; PAPER.md:94 quotes the
    threshold 3)."""
    f = np.asarray(f, float)
    N = f.shape[0] // 2
    a, b = birkhoff_average(f[:N]), birkhoff_average(f[N:2 * N])
    scale = max(abs(a), abs(b))
    d = abs(a - b)
    digits = 16.0 if (d == 0.0 or scale == 0.0) else min(16.0, -np.log10(d / scale))
    return a, b, float(digits)


# ---- orbit classification, characteristic frequencies, J_par from uniform-time samples -------------------------------
# "Given trajectory data, transport diagnostics include Poincare plots, characteristic orbit frequencies,
# weighted Birkhoff averaging (Duignan & Meiss, 2023), and orbit classification".  The paper prints no definition;
# reading A30 of DESIGN.md section 12, written out here on ONE particle's series sampled every dt:
#   * a reversal is a pair of consecutive samples with (v_j < 0) != (v_{j+1} < 0); its time is the zero of the straight
#     line through the two samples, tau = t_j + dt v_j / (v_j - v_{j+1});
#   * class 0 = passing (no reversal), 1 = trapped (at least one);
#   * omega_theta, omega_zeta = (angle_last - angle_first) / (t_last - t_first): the mean poloidal and toroidal rates;
#   * bounce frequency: with R >= 3 reversals, P = (R - 1) // 2 full periods lie between reversal 0 and reversal 2 P:
#     omega_b = 2 pi P / (tau_{2P} - tau_0); 0 otherwise;
#   * J_par of period p = m * integral of v_par^2 dt from tau_{2p} to tau_{2p+2} (dl = v_par dt along the orbit), by the
#     trapezoid rule on the samples in between, with v_par = 0 at both ends; reported: the mean over the P periods and
#     (max - min) / mean ("J_par and its variation").
def orbit_diagnostics(theta, zeta, vpar, dt: float, mass: float) -> dict:
    """theta, zeta, vpar: the valid samples of one particle (1-D arrays of equal length >= 2)."""
    theta, zeta, vpar = (np.asarray(a, float) for a in (theta, zeta, vpar))
    c = vpar.shape[0]
    nan = float("nan")
    if c < 2:
        return dict(orbit_class=nan, reversals=0, omega_theta=nan, omega_zeta=nan, omega_bounce=nan, j_par=nan,
                    j_par_variation=nan)
    T = (c - 1) * dt
    taus, idx = [], []
    for j in range(c - 1):
        if (vpar[j] < 0.0) != (vpar[j + 1] < 0.0):
            taus.append(j * dt + dt * vpar[j] / (vpar[j] - vpar[j + 1]))
            idx.append(j)
    R = len(taus)
    P = (R - 1) // 2 if R >= 3 else 0
    omega_b, jmean, jvar = 0.0, nan, nan
    if P > 0:
        omega_b = 2.0 * math.pi * P / (taus[2 * P] - taus[0])
        J = []
        for p in range(P):
            a, b = 2 * p, 2 * p + 2
            ja, jb = idx[a] + 1, idx[b]                       # first and last sample inside the period
            acc = 0.5 * vpar[ja] ** 2 * (ja * dt - taus[a])    # from the reversal (v = 0) to the first sample
            for j in range(ja, jb):
                acc += 0.5 * (vpar[j] ** 2 + vpar[j + 1] ** 2) * dt
            acc += 0.5 * vpar[jb] ** 2 * (taus[b] - jb * dt)   # from the last sample to the reversal
            J.append(mass * acc)
        jmean = sum(J) / P
        jvar = (max(J) - min(J)) / jmean
    return dict(orbit_class=1.0 if R >= 1 else 0.0, reversals=R, omega_theta=(theta[-1] - theta[0]) / T,
                omega_zeta=(zeta[-1] - zeta[0]) / T, omega_bounce=omega_b, j_par=jmean, j_par_variation=jvar)
