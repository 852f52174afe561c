"""Seeded synthetic inputs for the guiding-centre hot path (BASELINE.json:configs).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA path.  It holds the input *recipes*
only: harmonic lists, table values, profiles, mode tables and particle initial conditions.  It does not
evaluate the field, the guiding-centre equations or the integrator, and it imports neither side.

The paper's workloads run on equilibria that do not exist in this repository (Wistell-A, precise QA/QH;
PAPER.md:72,78,94).  The configurations below stand in for them, taking their shapes: 3.5 MeV alpha
particles, 1e-4..2e-2 s horizons, 5e2..1e6 markers, harmonics on a uniform radial grid,
single- and multi-harmonic shear-Alfven modes.  Readings A15, A16, A19-A22 of SURVEY.md
§8(c) fix what BASELINE.json leaves open; DESIGN.md lists them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field as _dc_field

import numpy as np

# --- physical constants of the configs (BASELINE.json:configs[0]) -------------------------------------
ALPHA_MASS = 6.64e-27                      # kg
ELEMENTARY_CHARGE = 1.602176634e-19        # C
ALPHA_CHARGE = 2.0 * ELEMENTARY_CHARGE     # C
ALPHA_ENERGY = 3.5e6 * ELEMENTARY_CHARGE   # J
V_ALPHA = math.sqrt(2.0 * ALPHA_ENERGY / ALPHA_MASS)   # m/s, = v_ref of every config (A11)
B00 = 5.7                                  # T
R0 = 10.0                                  # m
A_MINOR = 1.7                              # m
PSI0 = B00 * A_MINOR ** 2 / 2.0            # T m^2
NFP = 4


@dataclass
class Field:
    """Host-side tables of one synthetic equilibrium (+ optional modes).  Layouts as SURVEY.md §8(b)."""
    ns: int
    nfp: int
    xm: np.ndarray          # [nh] int32, m >= 0
    xn: np.ndarray          # [nh] int32, in units of nfp
    bmnc: np.ndarray        # [ns][nh] float64, tesla
    G: np.ndarray           # [ns]
    I: np.ndarray           # [ns]
    iota: np.ndarray        # [ns]
    psi0: float
    mode_m: np.ndarray = _dc_field(default_factory=lambda: np.zeros(0, np.int32))
    mode_n: np.ndarray = _dc_field(default_factory=lambda: np.zeros(0, np.int32))
    mode_omega: np.ndarray = _dc_field(default_factory=lambda: np.zeros(0))
    mode_phase: np.ndarray = _dc_field(default_factory=lambda: np.zeros(0))
    phihat: np.ndarray = _dc_field(default_factory=lambda: np.zeros((0, 0)))   # [ns][nk], volts
    # NEXT-4 of SURVEY.md section 8(f): tables that stellarator symmetry and the K = 0 reading leave out (None = absent)
    bmns: np.ndarray | None = None      # [ns][nh] sin coefficients of B
    kmnc: np.ndarray | None = None      # [ns][nh] cos coefficients of the covariant radial component K
    kmns: np.ndarray | None = None      # [ns][nh] sin coefficients of K

    @property
    def nh(self) -> int:
        return int(self.xm.shape[0])

    @property
    def nk(self) -> int:
        return int(self.mode_m.shape[0])


@dataclass
class Particles:
    """Initial conditions before mu is known: mu needs one field evaluation, which the caller does with
    the implementation under test ('same arrays to both')."""
    s: np.ndarray
    theta: np.ndarray
    zeta: np.ndarray
    pitch: np.ndarray       # v_par / v in [-1, 1]
    speed: np.ndarray       # m/s

    @property
    def n(self) -> int:
        return int(self.s.shape[0])

    @property
    def vpar(self) -> np.ndarray:
        return self.pitch * self.speed

    def vperp2(self) -> np.ndarray:
        return (1.0 - self.pitch ** 2) * self.speed ** 2

    def head(self, k: int) -> "Particles":
        return Particles(self.s[:k].copy(), self.theta[:k].copy(), self.zeta[:k].copy(),
                         self.pitch[:k].copy(), self.speed[:k].copy())


@dataclass
class TraceSpec:
    """Integrator specification of a config (O6 defaults)."""
    mass: float = ALPHA_MASS
    charge: float = ALPHA_CHARGE
    t0: float = 0.0
    t_max: float = 1e-4
    rtol: float = 1e-9
    atol: float = 1e-9
    v_ref: float = V_ALPHA
    h0: float = 1e-9
    h_min: float = 0.0
    s_loss: float = 1.0
    s_min: float = 1e-3
    max_steps: int = 2_000_000_000


def harmonic_list(M: int, N: int):
    """m = 0: n = 0..N; m = 1..M: n = -N..N (A20).  nh = (N+1) + M(2N+1): 145 for 8/8, 545 for 16/16."""
    xm, xn = [], []
    for m in range(M + 1):
        for n in range(0 if m == 0 else -N, N + 1):
            xm.append(m)
            xn.append(n)
    return np.asarray(xm, np.int32), np.asarray(xn, np.int32)


def make_equilibrium(M: int, N: int, ns: int, seed: int = 0, nfp: int = NFP) -> Field:
    """BASELINE.json:configs[0] field recipe with draw order A21."""
    xm, xn = harmonic_list(M, N)
    nh = xm.shape[0]
    rng = np.random.default_rng(seed)
    g = rng.standard_normal(nh)
    s = np.arange(ns, dtype=np.float64) / (ns - 1)
    amp = 0.05 * B00 * g * np.exp(-(xm + np.abs(xn)) / 3.0)              # [nh]
    bmnc = amp[None, :] * np.power(s[:, None], xm[None, :] / 2.0)         # s^{m/2}; 0^0 = 1
    bmnc[:, 0] = B00                                                      # (m, n) = (0, 0) overrides
    return Field(ns=ns, nfp=nfp, xm=xm, xn=xn, bmnc=np.ascontiguousarray(bmnc),
                 G=np.full(ns, B00 * R0), I=np.zeros(ns), iota=0.42 + 0.1 * s, psi0=PSI0)


def _alpha_hat_over_phi_hat(fld: Field, m: int, n: int, omega: float) -> np.ndarray:
    """Ratio alpha_hat/Phi_hat at the radial nodes used ONLY to scale a mode to its stated deltaB/B
    (A14, A16): -(iota m - n) / (omega (G + iota I))."""
    return -(fld.iota * m - n) / (omega * (fld.G + fld.iota * fld.I))


def _normalise_mode(fld: Field, ms, ns_, omegas, envelope: np.ndarray, dB_over_B: float) -> float:
    """Amplitude A (volts) so that max_s sqrt(sum_k (m_k alpha_hat_k / (a sqrt s))^2) = dB_over_B (A16)."""
    s = np.arange(fld.ns, dtype=np.float64) / (fld.ns - 1)
    tot = np.zeros(fld.ns)
    for m, n, w in zip(ms, ns_, omegas):
        ah = _alpha_hat_over_phi_hat(fld, int(m), int(n), float(w)) * envelope
        with np.errstate(divide="ignore", invalid="ignore"):
            r = np.where(s > 0, m * ah / (A_MINOR * np.sqrt(np.maximum(s, 1e-300))), 0.0)
        tot += r * r
    peak = math.sqrt(tot.max())
    return dB_over_B / peak


def add_single_ae(fld: Field) -> Field:
    """Config 2 (A15): one eigenmode, 8 harmonics m=3..6 x n=2..3, 120 kHz, Gaussian s_c=0.4, width 0.05,
    jointly normalised to deltaB/B = 1e-4."""
    s = np.arange(fld.ns, dtype=np.float64) / (fld.ns - 1)
    ms, ns_ = [], []
    for m in range(3, 7):
        for n in (2, 3):
            ms.append(m)
            ns_.append(n)
    K = len(ms)
    omega = np.full(K, 2.0 * math.pi * 120e3)
    env = np.exp(-((s - 0.4) ** 2) / (2.0 * 0.05 ** 2))
    A = _normalise_mode(fld, ms, ns_, omega, env, 1e-4)
    fld.mode_m = np.asarray(ms, np.int32)
    fld.mode_n = np.asarray(ns_, np.int32)
    fld.mode_omega = omega
    fld.mode_phase = np.zeros(K)
    fld.phihat = np.ascontiguousarray(np.repeat((A * env)[:, None], K, axis=1))
    return fld


def add_random_aes(fld: Field, K: int = 16, seed: int = 2004) -> Field:
    """Config 4 (A22): K single-harmonic modes; m~U{1..12}, n~U{-6..6}\\{0}, f~U[50,300] kHz,
    s_c~U[0.2,0.8], width 0.05, phase~U[0,2pi), deltaB/B = 5e-5 each."""
    rng = np.random.default_rng(seed)
    s = np.arange(fld.ns, dtype=np.float64) / (fld.ns - 1)
    m = rng.integers(1, 13, size=K)
    nz = rng.integers(1, 7, size=K) * rng.choice(np.array([-1, 1]), size=K)
    f = rng.uniform(50e3, 300e3, size=K)
    sc = rng.uniform(0.2, 0.8, size=K)
    ph = rng.uniform(0.0, 2.0 * math.pi, size=K)
    omega = 2.0 * math.pi * f
    phihat = np.zeros((fld.ns, K))
    for k in range(K):
        env = np.exp(-((s - sc[k]) ** 2) / (2.0 * 0.05 ** 2))
        A = _normalise_mode(fld, [m[k]], [nz[k]], [omega[k]], env, 5e-5)
        phihat[:, k] = A * env
    fld.mode_m = m.astype(np.int32)
    fld.mode_n = nz.astype(np.int32)
    fld.mode_omega = omega
    fld.mode_phase = ph
    fld.phihat = np.ascontiguousarray(phihat)
    return fld


def make_particles(config: int, n: int | None = None, stream: int = 0) -> Particles:
    """Initial conditions of BASELINE.json:configs[config]; draw order s, theta, zeta, pitch, speed (A21).
    ``n`` overrides the ensemble size; the first k particles of a larger draw are NOT the same as a draw
    of k, so subsamples are always taken with ``Particles.head`` from the full-size draw or drawn at the
    size the test states."""
    full = {0: 512, 1: 100_000, 2: 100_000, 3: 1_000_000, 4: 1_000_000}[config]
    n = full if n is None else int(n)
    # stream 0 is the ensemble of the config; stream r > 0 is an independent draw of the same recipe (one
    # per rank of a weak-scaling run)
    rng = np.random.default_rng(1000 + config if stream == 0 else [1000 + config, int(stream)])
    if config == 0:
        s = np.full(n, 0.25)
    elif config in (1, 2):
        s = rng.uniform(0.1, 0.5, size=n)
    else:
        s = 1.0 - np.cbrt(1.0 - rng.uniform(0.0, 1.0, size=n))            # pdf (1-s)^2 (A19)
    theta = rng.uniform(0.0, 2.0 * math.pi, size=n)
    zeta = rng.uniform(0.0, 2.0 * math.pi, size=n)
    pitch = rng.uniform(-1.0, 1.0, size=n)
    if config in (3, 4):
        vc = 0.3 * V_ALPHA
        U = rng.uniform(0.0, 1.0, size=n)
        speed = vc * np.cbrt(np.expm1(U * math.log1p((V_ALPHA / vc) ** 3)))  # slowing-down speeds (A19)
    else:
        speed = np.full(n, V_ALPHA)
    return Particles(s, theta, zeta, pitch, speed)


def make_field(config: int) -> Field:
    if config == 0:
        return make_equilibrium(8, 8, 51)
    fld = make_equilibrium(16, 16, 101)
    if config == 2:
        add_single_ae(fld)
    elif config == 4:
        add_random_aes(fld)
    return fld


def make_spec(config: int) -> TraceSpec:
    return {
        0: TraceSpec(t_max=1e-4, rtol=1e-9, atol=1e-9),
        1: TraceSpec(t_max=1e-2, rtol=1e-9, atol=1e-9, h_min=1e-12),
        2: TraceSpec(t_max=5e-3, rtol=1e-9, atol=1e-9),
        3: TraceSpec(t_max=2e-2, rtol=1e-8, atol=1e-8),
        4: TraceSpec(t_max=1e-2, rtol=1e-9, atol=1e-9),
    }[config]


def mu_from(particles: Particles, B_at_start: np.ndarray, mass: float = ALPHA_MASS) -> np.ndarray:
    """mu = m v_perp^2 / (2 B) in J/T (A5); ``B_at_start`` comes from the implementation under test."""
    return 0.5 * mass * particles.vperp2() / B_at_start
