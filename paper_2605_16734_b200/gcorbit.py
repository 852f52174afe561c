"""Thin Python binding of libgcorbit.so (include/gcorbit.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for device memory and
streams, nothing else.  There is no CPU fallback: if the library is missing or no CUDA device is present the
calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(_HERE, "libgcorbit.so")

GC_OK, GC_EINVAL, GC_ENOMEM, GC_ECUDA = 0, -1, -2, -3
GC_KERNEL_AUTO, GC_KERNEL_GENERIC, GC_KERNEL_WARP, GC_KERNEL_TILE, GC_KERNEL_MMA, GC_KERNEL_GRID = 0, 1, 2, 3, 4, 5
GC_TILE_MIN_PARTICLES, GC_TILE_MIN_PARTICLES_SMALL = 3072, 2048
GC_OPT_WAVE_PARTICLES, GC_OPT_CHUNK_ATTEMPTS = 1, 2
GC_GRID_LAGRANGE, GC_GRID_HERMITE = 0, 1
ST_TMAX, ST_LOST, ST_AXIS, ST_MAXSTEPS, ST_NONFINITE = 0, 1, 2, 3, 4

EXPORTS = ["gc_field_create", "gc_field_destroy", "gc_field_eval", "gc_pert_eval", "gc_rhs_eval", "gc_trace",
           "gc_trace_host", "gc_set_kernel", "gc_set_option", "gc_kernel_info", "gc_last_error",
           "gc_trace_sampled", "gc_pzeta_eval", "gc_birkhoff", "gc_kcov_eval", "gc_field_set_grid", "gc_trace_symplectic", "gc_orbit_diagnostics",
           "gc_trace_noalloc"]


class GcError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"gcorbit error {code}: {msg}")
        self.code = code


class gc_field_desc(C.Structure):
    _fields_ = [("ns", C.c_int32), ("nfp", C.c_int32), ("nh", C.c_int32),
                ("xm", C.c_void_p), ("xn", C.c_void_p), ("bmnc", C.c_void_p),
                ("G", C.c_void_p), ("I", C.c_void_p), ("iota", C.c_void_p),
                ("psi0", C.c_double), ("nk", C.c_int32),
                ("mode_m", C.c_void_p), ("mode_n", C.c_void_p),
                ("mode_omega", C.c_void_p), ("mode_phase", C.c_void_p), ("phihat", C.c_void_p),
                ("bmns", C.c_void_p), ("kmnc", C.c_void_p), ("kmns", C.c_void_p)]


class gc_trace_params(C.Structure):
    _fields_ = [("mass", C.c_double), ("charge", C.c_double), ("t0", C.c_double), ("t_max", C.c_double),
                ("rtol", C.c_double), ("atol", C.c_double), ("v_ref", C.c_double),
                ("h0", C.c_double), ("h_min", C.c_double), ("s_loss", C.c_double), ("s_min", C.c_double),
                ("max_steps", C.c_int64), ("poincare_capacity", C.c_int64), ("flags", C.c_int64)]


_lib = None


def load_library():
    """dlopen libgcorbit.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO_PATH):
            raise FileNotFoundError(f"{SO_PATH} not built: run `python __graft_entry__.py build` "
                                    "(no CPU fallback exists)")
        L = C.CDLL(SO_PATH)
        vp, i64, dbl, i32 = C.c_void_p, C.c_int64, C.c_double, C.c_int32
        L.gc_last_error.restype = C.c_char_p
        L.gc_field_create.argtypes = [C.POINTER(gc_field_desc), C.POINTER(vp)]
        L.gc_field_destroy.argtypes = [vp]
        L.gc_field_eval.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp]
        L.gc_kcov_eval.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp]
        L.gc_pert_eval.argtypes = [vp, i64, vp, vp, vp, dbl, vp, vp]
        L.gc_rhs_eval.argtypes = [vp, dbl, dbl, dbl, i64, vp, vp, vp, vp]
        L.gc_trace.argtypes = [vp, C.POINTER(gc_trace_params), i64] + [vp] * 15
        L.gc_trace_noalloc.argtypes = [vp, C.POINTER(gc_trace_params), i64] + [vp] * 15
        L.gc_trace_host.argtypes = [vp, C.POINTER(gc_trace_params), i64] + [vp] * 14
        L.gc_trace_sampled.argtypes = [vp, C.POINTER(gc_trace_params), i64] + [vp] * 12 + [dbl, dbl, i64, vp, vp, vp]
        L.gc_pzeta_eval.argtypes = [vp, dbl, dbl, i64, vp, vp, vp, vp, vp]
        L.gc_birkhoff.argtypes = [i64, i64, vp, i64, vp, vp, vp]
        L.gc_set_kernel.argtypes = [vp, i32]
        L.gc_orbit_diagnostics.argtypes = [i64, i64, vp, i64, vp, dbl, dbl, vp, vp]
        L.gc_field_set_grid.argtypes = [vp, i32, i32, i32, i32, vp]
        L.gc_trace_symplectic.argtypes = [vp, C.POINTER(gc_symplectic_params), i64] + [vp] * 11 + [i64, i64, vp, vp, vp]
        L.gc_set_option.argtypes = [vp, i32, i64]
        L.gc_kernel_info.argtypes = [vp, C.c_int64] + [C.POINTER(i32)] * 5
        for name in EXPORTS:
            if name != "gc_last_error":
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _check(rc: int):
    if rc != GC_OK:
        raise GcError(rc, load_library().gc_last_error().decode())


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("gcorbit needs a CUDA device; there is no CPU fallback")
    return torch


def _hp(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _dp(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream_ptr(torch):
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


NOALLOC_MAX_PARTICLES = 32768      # GC_NOALLOC_MAX_PARTICLES of include/gcorbit.h
GC_TRACE_RESUME = 1
GC_TRACE_SECTION_VPAR = 2
GC_TRACE_REFINE_LOSS = 4


def make_params(spec, t0=None, t_max=None, poincare_capacity=0, flags=0) -> gc_trace_params:
    return gc_trace_params(spec.mass, spec.charge, spec.t0 if t0 is None else t0,
                           spec.t_max if t_max is None else t_max, spec.rtol, spec.atol, spec.v_ref,
                           spec.h0, spec.h_min, spec.s_loss, spec.s_min, int(spec.max_steps),
                           int(poincare_capacity), int(flags))


@dataclass
class TraceResult:
    y: object            # [4][n]: s, theta, zeta, v_par (m/s)
    t: object            # [n]
    status: object       # [n] int32
    n_acc: object
    n_rej: object
    n_forced: object
    h: object            # [n]
    poincare: object = None
    poincare_count: int = 0
    samples: object = None        # [4][nsamp][n] (gc_trace_sampled)
    sample_end: object = None     # [n] int32


def orbit_diagnostics(samples, j_first, sample_end, sample_dt, mass):
    """gc_orbit_diagnostics: samples [4][nsamp][n] device tensor -> out [7][n] (class, reversals, omega_theta,
    omega_zeta, omega_bounce, J_par, J_par variation)."""
    torch = _torch()
    _, nsamp, n = samples.shape
    assert samples.is_contiguous()
    out = torch.empty((7, n), dtype=torch.float64, device=samples.device)
    _check(load_library().gc_orbit_diagnostics(n, nsamp, _dp(samples), int(j_first), _dp(sample_end), float(sample_dt),
                                               float(mass), _dp(out), _stream_ptr(torch)))
    return out


class gc_symplectic_params(C.Structure):
    _fields_ = [("mass", C.c_double), ("charge", C.c_double), ("t0", C.c_double), ("dt", C.c_double),
                ("nsteps", C.c_int64), ("s_loss", C.c_double), ("s_min", C.c_double), ("newton_tol", C.c_double),
                ("max_iter", C.c_int64), ("flags", C.c_int64)]


@dataclass
class SymplecticResult:
    y: object            # [4][n]: s, theta, zeta, v_par (m/s)
    t: object            # [n]
    status: object       # [n] int32
    n_steps: object
    n_iter: object
    samples: object = None        # [4][nsamp][n]
    sample_end: object = None


class Field:
    """gc_field_create / gc_field_destroy.  ``fld`` carries host numpy tables (workloads.Field layout)."""

    def __init__(self, fld):
        L = load_library()
        k = dict(xm=np.ascontiguousarray(fld.xm, np.int32), xn=np.ascontiguousarray(fld.xn, np.int32),
                 bmnc=np.ascontiguousarray(fld.bmnc, np.float64), G=np.ascontiguousarray(fld.G, np.float64),
                 I=np.ascontiguousarray(fld.I, np.float64), iota=np.ascontiguousarray(fld.iota, np.float64),
                 mode_m=np.ascontiguousarray(fld.mode_m, np.int32),
                 mode_n=np.ascontiguousarray(fld.mode_n, np.int32),
                 mode_omega=np.ascontiguousarray(fld.mode_omega, np.float64),
                 mode_phase=np.ascontiguousarray(fld.mode_phase, np.float64),
                 phihat=np.ascontiguousarray(fld.phihat, np.float64))
        ns, nh, nk = int(fld.ns), int(k["xm"].shape[0]), int(k["mode_m"].shape[0])
        for name in ("bmns", "kmnc", "kmns"):                  # NEXT-4 tables: None = absent
            a = getattr(fld, name, None)
            k[name] = None if a is None else np.ascontiguousarray(a, np.float64)
        if k["bmnc"].shape != (ns, nh) or (nk and k["phihat"].shape != (ns, nk)) or \
                any(k[nm] is not None and k[nm].shape != (ns, nh) for nm in ("bmns", "kmnc", "kmns")):
            raise ValueError("table shapes do not match ns, nh, nk")
        d = gc_field_desc(ns, int(fld.nfp), nh, _hp(k["xm"]), _hp(k["xn"]), _hp(k["bmnc"]), _hp(k["G"]),
                          _hp(k["I"]), _hp(k["iota"]), float(fld.psi0), nk, _hp(k["mode_m"]),
                          _hp(k["mode_n"]), _hp(k["mode_omega"]), _hp(k["mode_phase"]), _hp(k["phihat"]),
                          _hp(k["bmns"]), _hp(k["kmnc"]), _hp(k["kmns"]))
        h = C.c_void_p(None)
        _check(L.gc_field_create(C.byref(d), C.byref(h)))
        self._h = h
        self.ns, self.nh, self.nk = ns, nh, nk

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().gc_field_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- gc_set_kernel / gc_kernel_info --------------------------------------------------------------------
    def set_kernel(self, kernel: int):
        _check(load_library().gc_set_kernel(self._h, kernel))

    def set_option(self, option: int, value: int):
        _check(load_library().gc_set_option(self._h, int(option), int(value)))

    def set_grid(self, ngs: int, nth: int, nze: int, kind: int = 0):
        """gc_field_set_grid (NEXT-2): B becomes a tricubic interpolant of its node values (kind GC_GRID_LAGRANGE) or
        of its node values and derivatives (GC_GRID_HERMITE); (0, 0, 0) drops it."""
        torch = _torch()
        _check(load_library().gc_field_set_grid(self._h, int(ngs), int(nth), int(nze), int(kind), _stream_ptr(torch)))

    def kernel_info(self, n: int = 1 << 20) -> dict:
        """Kernel and launch geometry gc_trace uses for an ensemble of n particles."""
        v = [C.c_int32(0) for _ in range(5)]
        _check(load_library().gc_kernel_info(self._h, int(n), *[C.byref(x) for x in v]))
        return dict(kernel={GC_KERNEL_GENERIC: "generic", GC_KERNEL_WARP: "warp", GC_KERNEL_TILE: "tile", GC_KERNEL_MMA: "mma",
                            GC_KERNEL_GRID: "grid"}[v[0].value],
                    blocks=v[1].value, threads=v[2].value, smem_bytes=v[3].value, regs=v[4].value)

    # ---- gc_field_eval / gc_pert_eval / gc_rhs_eval (device tensors in, device tensors out) ------------------
    def field_eval(self, s, th, ze, derivs=True):
        torch = _torch()
        n = s.numel()
        B = torch.empty(n, dtype=torch.float64, device=s.device)
        dB = torch.empty((3, n), dtype=torch.float64, device=s.device) if derivs else None
        _check(load_library().gc_field_eval(self._h, n, _dp(s), _dp(th), _dp(ze), _dp(B), _dp(dB),
                                            _stream_ptr(torch)))
        return B, dB

    def kcov_eval(self, s, th, ze, derivs=True):
        torch = _torch()
        n = s.numel()
        K = torch.empty(n, dtype=torch.float64, device=s.device)
        dK = torch.empty((3, n), dtype=torch.float64, device=s.device) if derivs else None
        _check(load_library().gc_kcov_eval(self._h, n, _dp(s), _dp(th), _dp(ze), _dp(K), _dp(dK), _stream_ptr(torch)))
        return K, dK

    def pert_eval(self, s, th, ze, t):
        torch = _torch()
        n = s.numel()
        out = torch.empty((9, n), dtype=torch.float64, device=s.device)
        _check(load_library().gc_pert_eval(self._h, n, _dp(s), _dp(th), _dp(ze), float(t), _dp(out),
                                           _stream_ptr(torch)))
        return out

    def rhs_eval(self, mass, charge, t, y, mu):
        torch = _torch()
        n = mu.numel()
        assert y.shape == (4, n) and y.is_contiguous()
        out = torch.empty((4, n), dtype=torch.float64, device=y.device)
        _check(load_library().gc_rhs_eval(self._h, float(mass), float(charge), float(t), n, _dp(y), _dp(mu),
                                          _dp(out), _stream_ptr(torch)))
        return out

    # ---- gc_trace (device tensors) ---------------------------------------------------------------------------
    def trace(self, spec, s0, th0, ze0, vpar0, mu, h_inout=None, poincare_capacity=0, t0=None, t_max=None,
              counters=True, out=None, flags=0) -> TraceResult:
        """Asynchronous on torch's current stream.  ``out`` may carry a previous TraceResult whose buffers are
        reused (no allocation inside a timed region)."""
        torch = _torch()
        n = s0.numel()
        dev = s0.device
        for x in (s0, th0, ze0, vpar0, mu):
            assert x.dtype == torch.float64 and x.is_cuda and x.is_contiguous() and x.numel() == n
        p = make_params(spec, t0, t_max, poincare_capacity, flags)
        if out is None:
            i32 = lambda: torch.empty(n, dtype=torch.int32, device=dev)
            out = TraceResult(torch.empty((4, n), dtype=torch.float64, device=dev),
                              torch.empty(n, dtype=torch.float64, device=dev), i32(),
                              i32() if counters else None, i32() if counters else None,
                              i32() if counters else None, h_inout)
            if poincare_capacity:
                out.poincare = torch.empty((poincare_capacity, 4), dtype=torch.float64, device=dev)
        out.h = h_inout
        cnt = torch.zeros(1, dtype=torch.int64, device=dev) if poincare_capacity else None
        _check(load_library().gc_trace(self._h, C.byref(p), n, _dp(s0), _dp(th0), _dp(ze0), _dp(vpar0), _dp(mu),
                                       _dp(h_inout), _dp(out.y), _dp(out.t), _dp(out.status), _dp(out.n_acc),
                                       _dp(out.n_rej), _dp(out.n_forced),
                                       _dp(out.poincare) if poincare_capacity else None, _dp(cnt),
                                       _stream_ptr(torch)))
        out._count_tensor = cnt
        return out

    # ---- gc_trace_noalloc (device tensors) -------------------------------------------------------------------
    def trace_noalloc(self, spec, s0, th0, ze0, vpar0, mu, out: TraceResult, h_inout=None, t0=None, t_max=None,
                      flags=0, poincare_count=None) -> TraceResult:
        """gc_trace for hosts that must not allocate on the GPU while they run (a service whose own arena owns the
        device, a loop with a deadline, a plug-in under a foreign allocator): the library works in a fixed 5 MiB
        array inside its own image instead of pool memory.  At most ``NOALLOC_MAX_PARTICLES`` particles per call;
        calls share the one array, so keep them on one stream.  Nothing is allocated here either: ``out`` must
        carry every output buffer (y, t, status; counters and poincare if wanted), and Poincare records need the
        caller's one-element int64 ``poincare_count`` tensor.  Asynchronous on torch's current stream."""
        torch = _torch()
        n = s0.numel()
        for x in (s0, th0, ze0, vpar0, mu):
            assert x.dtype == torch.float64 and x.is_cuda and x.is_contiguous() and x.numel() == n
        cap = 0 if out.poincare is None or poincare_count is None else out.poincare.shape[0]
        p = make_params(spec, t0, t_max, cap, flags)
        out.h = h_inout
        _check(load_library().gc_trace_noalloc(self._h, C.byref(p), n, _dp(s0), _dp(th0), _dp(ze0), _dp(vpar0),
                                               _dp(mu), _dp(h_inout), _dp(out.y), _dp(out.t), _dp(out.status),
                                               _dp(out.n_acc), _dp(out.n_rej), _dp(out.n_forced),
                                               _dp(out.poincare) if cap else None,
                                               _dp(poincare_count) if cap else None, _stream_ptr(torch)))
        out._count_tensor = poincare_count if cap else None
        return out

    # ---- NEXT-1: gc_trace_sampled / gc_pzeta_eval / gc_birkhoff ----------------------------------------------------
    def trace_sampled(self, spec, s0, th0, ze0, vpar0, mu, sample_t0, sample_dt, nsamp, h_inout=None, t0=None,
                      t_max=None, out=None, flags=0) -> TraceResult:
        """gc_trace plus uniform-time samples of the continuous extension (O9).  ``out`` may carry the result of a
        previous call (same sample buffers: the grid continues under GC_TRACE_RESUME)."""
        torch = _torch()
        n = s0.numel()
        dev = s0.device
        p = make_params(spec, t0, t_max, 0, flags)
        if out is None:
            i32 = lambda: torch.empty(n, dtype=torch.int32, device=dev)
            out = TraceResult(torch.empty((4, n), dtype=torch.float64, device=dev),
                              torch.empty(n, dtype=torch.float64, device=dev), i32(), i32(), i32(), i32(), h_inout)
            out.samples = torch.full((4, int(nsamp), n), float("nan"), dtype=torch.float64, device=dev)
            out.sample_end = torch.zeros(n, dtype=torch.int32, device=dev)
        out.h = h_inout
        _check(load_library().gc_trace_sampled(self._h, C.byref(p), n, _dp(s0), _dp(th0), _dp(ze0), _dp(vpar0),
                                               _dp(mu), _dp(h_inout), _dp(out.y), _dp(out.t), _dp(out.status),
                                               _dp(out.n_acc), _dp(out.n_rej), _dp(out.n_forced), float(sample_t0),
                                               float(sample_dt), int(nsamp), _dp(out.samples), _dp(out.sample_end),
                                               _stream_ptr(torch)))
        return out

    def pzeta_eval(self, mass, charge, y, t, chi_nodes):
        """P_zeta at the n states y [4][n] (device) and times t [n] (device or None); chi_nodes [ns] device."""
        torch = _torch()
        n = y.shape[1]
        out = torch.empty(n, dtype=torch.float64, device=y.device)
        _check(load_library().gc_pzeta_eval(self._h, float(mass), float(charge), n, _dp(y), _dp(t), _dp(chi_nodes),
                                            _dp(out), _stream_ptr(torch)))
        return out

    def trace_symplectic(self, mass, charge, s0, th0, ze0, vpar0, mu, chi_nodes, dt, nsteps, t0=0.0, s_loss=1.0,
                         s_min=1e-3, newton_tol=1e-13, max_iter=50, sample_stride=0, nsamp=0, out=None, flags=0):
        """gc_trace_symplectic (NEXT-3).  Returns a SymplecticResult of device tensors; ``out`` may carry the result
        of a previous call (buffers reused; with GC_TRACE_RESUME the call continues it in place)."""
        torch = _torch()
        n = s0.numel()
        dev = s0.device
        if out is None:
            out = SymplecticResult(torch.empty((4, n), dtype=torch.float64, device=dev),
                                   torch.empty(n, dtype=torch.float64, device=dev),
                                   torch.zeros(n, dtype=torch.int32, device=dev),
                                   torch.zeros(n, dtype=torch.int32, device=dev),
                                   torch.zeros(n, dtype=torch.int32, device=dev),
                                   torch.full((4, int(nsamp), n), float("nan"), dtype=torch.float64, device=dev)
                                   if nsamp else None,
                                   torch.zeros(n, dtype=torch.int32, device=dev) if nsamp else None)
        p = gc_symplectic_params(float(mass), float(charge), float(t0), float(dt), int(nsteps), float(s_loss),
                                 float(s_min), float(newton_tol), int(max_iter), int(flags))
        _check(load_library().gc_trace_symplectic(
            self._h, C.byref(p), C.c_int64(n), _dp(s0), _dp(th0), _dp(ze0), _dp(vpar0), _dp(mu), _dp(chi_nodes),
            _dp(out.y), _dp(out.t), _dp(out.status), _dp(out.n_steps), _dp(out.n_iter), C.c_int64(int(sample_stride)),
            C.c_int64(int(nsamp)), _dp(out.samples), _dp(out.sample_end), _stream_ptr(torch)))
        return out

    def trace_resume(self, spec, state: TraceResult, mu, t0, t_max, poincare_capacity=0) -> TraceResult:
        """Continue a previous ``trace`` result in place over [t0, t_max] (GC_TRACE_RESUME): the rows of
        ``state.y`` are the initial conditions and receive the new states; ``state.h`` carries the step
        proposals; particles whose status is not 0 are left untouched."""
        if state.h is None:
            raise ValueError("trace_resume needs the h_inout buffer of the first call")
        y = state.y
        return self.trace(spec, y[0], y[1], y[2], y[3], mu, h_inout=state.h,
                          poincare_capacity=poincare_capacity, t0=t0, t_max=t_max, out=state,
                          flags=GC_TRACE_RESUME)

    # ---- gc_trace_host (numpy in, numpy out; copies inside the call) --------------------------------------------
    def trace_host(self, spec, s0, th0, ze0, vpar0, mu, h_in=None, poincare_capacity=0, t0=None, t_max=None,
                   bufs=None, flags=0) -> TraceResult:
        """Host numpy arrays in and out (views of pinned torch tensors make the copies asynchronous).  With
        ``bufs`` given its arrays are the output buffers; under GC_TRACE_RESUME they are also read, ``bufs.h``
        is the h_inout array and the inputs may be the rows of ``bufs.y``."""
        chk = lambda a: a if (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous) \
            else np.ascontiguousarray(a, np.float64)
        s0, th0, ze0, vpar0, mu = map(chk, (s0, th0, ze0, vpar0, mu))
        n = s0.shape[0]
        p = make_params(spec, t0, t_max, poincare_capacity, flags)
        if bufs is None:
            bufs = TraceResult(np.empty((4, n)), np.empty(n), np.zeros(n, np.int32), np.zeros(n, np.int32),
                               np.zeros(n, np.int32), np.zeros(n, np.int32), None)
        if not (flags & GC_TRACE_RESUME) or bufs.h is None:
            bufs.h = np.zeros(n) if h_in is None else chk(h_in).copy()
        pc = np.empty((max(poincare_capacity, 1), 4)) if poincare_capacity else None
        cnt = C.c_int64(0)
        _check(load_library().gc_trace_host(self._h, C.byref(p), n, _hp(s0), _hp(th0), _hp(ze0), _hp(vpar0),
                                            _hp(mu), _hp(bufs.h), _hp(bufs.y), _hp(bufs.t), _hp(bufs.status),
                                            _hp(bufs.n_acc), _hp(bufs.n_rej), _hp(bufs.n_forced), _hp(pc),
                                            C.cast(C.byref(cnt), C.c_void_p) if poincare_capacity else None))
        if poincare_capacity:
            bufs.poincare_count = int(cnt.value)
            bufs.poincare = pc[:min(bufs.poincare_count, poincare_capacity)]
        return bufs


def finish_poincare(res: TraceResult) -> TraceResult:
    """After a stream synchronisation: read the device crossing counter of a ``Field.trace`` result."""
    cnt = getattr(res, "_count_tensor", None)
    if cnt is not None:
        res.poincare_count = int(cnt.item())
        res.poincare = res.poincare[:min(res.poincare_count, res.poincare.shape[0])]
    return res


def birkhoff(series, j_first=0, sample_end=None):
    """gc_birkhoff: series [nsamp][n] device tensor -> [3][n] (WB first half, WB second half, digit accuracy)."""
    torch = _torch()
    nsamp, n = series.shape
    out = torch.empty((3, n), dtype=torch.float64, device=series.device)
    _check(load_library().gc_birkhoff(n, nsamp, _dp(series), int(j_first), _dp(sample_end), _dp(out),
                                      _stream_ptr(torch)))
    return out
