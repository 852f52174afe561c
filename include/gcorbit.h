/* gcorbit.h -- C ABI of the B200 guiding-centre orbit tracer (libgcorbit.so, sm_100a, FP64).
 *
 * The boundary follows the paper's statement of the problem: "Integration of guiding center trajectories
 * is performed given the magnetic field, particle initial conditions, and integrator specification"
 * (section "Structure and capabilities").  The field is a set of Fourier harmonics on a
 * uniform radial grid evaluated by Lagrange interpolation, optionally with a superimposed MHD-mode
 * perturbation stored as a radial grid of Fourier harmonics; the integrator is a
 * Dormand-Prince 5 scheme with minimum-step control; particles are independent
 * (PAPER.md:48).  Where the paper prints no mathematics the operations are those of DESIGN.md section 2
 * (readings O1-O8, A1-A22 of SURVEY.md section 8(c)).
 *
 * Conventions.  Every function returns GC_OK (0) or a negative gc_status; the text of the last failure
 * on the calling thread is available from gc_last_error().  No C++ exception crosses the boundary.
 * The library never frees or retains caller buffers.  There is no CPU fallback: every entry point that
 * computes needs a CUDA device and fails with GC_ECUDA otherwise.
 */
#ifndef GCORBIT_H
#define GCORBIT_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  GC_OK = 0,
  GC_EINVAL = -1,   /* bad shape, NULL where data is required, NaN in a table, ns < 4, omega == 0 ... */
  GC_ENOMEM = -2,   /* host or device allocation failed                                               */
  GC_ECUDA = -3     /* CUDA runtime error; gc_last_error() carries cudaGetErrorString                 */
} gc_status;

typedef struct gc_field gc_field;   /* opaque; owns the device copies of all tables */

/* Field description.  ALL POINTERS ARE HOST MEMORY and are copied by gc_field_create.
 *   B(s,th,ze) = sum_k bmnc[.][k](s) cos(xm[k] th - xn[k] nfp ze)          stellarator-symmetric
 *   radial grid s_j = j/(ns-1), j = 0..ns-1; cubic (4-point) Lagrange interpolation in s (O1)
 *   perturbation  Phi = sum_k phihat[.][k](s) sin(mode_m th - mode_n ze + mode_omega t + mode_phase),
 *   alpha from Phi by the ideal-MHD constraint E_par = 0 (O3).
 * NEXT-4 of SURVEY.md section 8(f) (the field model of PAPER.md:44 without stellarator symmetry and with the covariant
 * radial component kept); each of the three tables may be NULL (= zero):
 *   B += sum_k bmns[.][k](s) sin(xm[k] th - xn[k] nfp ze)
 *   K  = sum_k kmnc[.][k](s) cos(xm[k] th - xn[k] nfp ze) + kmns[.][k](s) sin(...)   in B = G grad zeta + I grad theta
 *        + K grad psi; with K the equations of motion are the general Euler-Lagrange form.
 * Fields with any of the three are traced by the mma kernel (large ensembles) or the generic kernel.
 * Harmonic lists may come in any order; duplicate (m, n) pairs add.  Requires xm >= 0. */
typedef struct {
  int32_t ns;                 /* radial nodes, >= 4                                             */
  int32_t nfp;                /* field periods, >= 1                                            */
  int32_t nh;                 /* equilibrium harmonics, >= 1                                    */
  const int32_t* xm;          /* [nh] poloidal mode numbers, >= 0                               */
  const int32_t* xn;          /* [nh] toroidal mode numbers in units of nfp                     */
  const double* bmnc;         /* [ns][nh] node-major, tesla                                     */
  const double* G;            /* [ns] T m  (covariant toroidal component)                       */
  const double* I;            /* [ns] T m  (covariant poloidal component)                       */
  const double* iota;         /* [ns] rotational transform                                      */
  double psi0;                /* psi = psi0 * s: toroidal flux / 2 pi at s = 1, T m^2, != 0     */
  int32_t nk;                 /* perturbation harmonics; 0 = static field                       */
  const int32_t* mode_m;      /* [nk]                                                           */
  const int32_t* mode_n;      /* [nk] actual toroidal numbers                                   */
  const double* mode_omega;   /* [nk] rad/s, nonzero                                            */
  const double* mode_phase;   /* [nk] rad                                                       */
  const double* phihat;       /* [ns][nk] node-major, volts                                     */
  const double* bmns;         /* [ns][nh] node-major sin coefficients of B, tesla, or NULL      */
  const double* kmnc;         /* [ns][nh] node-major cos coefficients of K, 1/m (T m / (T m^2)), or NULL */
  const double* kmns;         /* [ns][nh] node-major sin coefficients of K, or NULL             */
} gc_field_desc;

/* Integrator specification (O5-O8).  The state integrated is (s, theta, zeta, v_par/v_ref). */
typedef struct {
  double mass, charge;        /* kg, C                                                          */
  double t0, t_max;           /* s                                                              */
  double rtol, atol;          /* RMS error norm, sk_i = atol + rtol max(|y_i|, |y_new_i|)       */
  double v_ref;               /* m/s, > 0: scale of v_par in the error norm (A11)               */
  double h0, h_min;           /* s; h0 > 0 first trial step; h_min >= 0 (0 disables the rule)   */
  double s_loss, s_min;       /* stop when s >= s_loss (lost) or s <= s_min (axis)              */
  int64_t max_steps;          /* attempted steps per particle before status 3                   */
  int64_t poincare_capacity;  /* records available in `poincare`; 0 disables recording (O8)     */
  int64_t flags;              /* GC_TRACE_* bits, 0 = none                                      */
} gc_trace_params;

/* gc_trace_params.flags.  GC_TRACE_RESUME: `status` is read on entry and only particles whose status is
 * GC_ST_TMAX (0) are traced, from (s0, th0, ze0, vpar0) at t0; every output of the others is left as it
 * is, and n_acc, n_rej, n_forced are added to instead of overwritten (max_steps stays per call).  Together with h_inout, and with s0..vpar0 aliasing the rows of y_out (allowed: a particle is read
 * once before anything of it is written), a long horizon runs as consecutive calls on the same buffers,
 * each continuing where the last one stopped (checkpoint / resume).
 * GC_TRACE_SECTION_VPAR (NEXT-1, O8b; "trapped particle Poincare map"): the Poincare records are taken
 * where v_par changes sign (the bounce points, both directions) instead of at zeta = 0 mod 2 pi; same record
 * format; small ensembles are then traced by the generic kernel.
 * GC_TRACE_REFINE_LOSS (O7b, the alternative reading of A8): a lost particle reports the point where the continuous
 * extension of its last step crosses s_loss (t_out, y_out; |s - s_loss| < 1e-13) instead of the end of that step;
 * step counts, samples and Poincare records are unchanged; small ensembles go to the generic kernel. */
enum { GC_TRACE_RESUME = 1, GC_TRACE_SECTION_VPAR = 2, GC_TRACE_REFINE_LOSS = 4 };

/* Per-particle exit status written by gc_trace. */
enum { GC_ST_TMAX = 0, GC_ST_LOST = 1, GC_ST_AXIS = 2, GC_ST_MAXSTEPS = 3, GC_ST_NONFINITE = 4 };

/* Kernel selection for gc_trace (gc_set_kernel).
 *   GC_KERNEL_MMA     cell-binned, one lane per particle, the harmonic sum as FP64 DMMA.8x8x4 over groups of eight
 *                     particles, stencil window staged in shared memory by bulk copy; the default for large
 *                     ensembles (needs max |xn| <= 16, max xm <= 16)
 *   GC_KERNEL_TILE    cell-binned, one thread per particle, stencil window staged in shared memory by bulk
 *                     copy; the kernel for large ensembles (needs max |xn| <= 16 and a window that fits
 *                     shared memory)
 *   GC_KERNEL_WARP    one warp per particle, stencil window in registers; the kernel for small ensembles
 *                     (needs max |xn| <= 16, max xm <= 28)
 *   GC_KERNEL_GENERIC one thread per particle, tables read from global memory; any field
 *   GC_KERNEL_GRID    one lane per particle, atomic particle queue, B from the 3-D interpolant of gc_field_set_grid;
 *                     reported by gc_kernel_info while a grid is set, not selectable through gc_set_kernel
 *   GC_KERNEL_AUTO    per call: MMA (else TILE) when the field fits it and n >= GC_TILE_MIN_PARTICLES (measured
 *                     switch-over, profiles/r2_ensemble_size_sweep.md; GC_TILE_MIN_PARTICLES_SMALL for fields with
 *                     max xm, max |xn| <= 8, whose warp kernel saturates earlier), else WARP
 *                     when the field fits it, else GENERIC.
 * All four implement the same equations and controller; their results differ at rounding level only. */
enum { GC_KERNEL_AUTO = 0, GC_KERNEL_GENERIC = 1, GC_KERNEL_WARP = 2, GC_KERNEL_TILE = 3, GC_KERNEL_MMA = 4, GC_KERNEL_GRID = 5 };
enum { GC_TILE_MIN_PARTICLES = 3072, GC_TILE_MIN_PARTICLES_SMALL = 2048 };

/* Copies the tables to the device, checks them (finite values, xm >= 0, omega != 0) and builds the packed layouts of
 * every trace kernel the field fits: the by-node lane rows of the warp kernel, the per-cell window images of the
 * tile kernel and the by-node DMMA-fragment image of the mma kernel.  *out is NULL on
 * failure. */
int gc_field_create(const gc_field_desc* desc, gc_field** out);
int gc_field_destroy(gc_field* f);

/* ---- NEXT-2 of SURVEY.md section 8(f): the 3-D local-interpolant field ("CUDA kernels implement field interpolation
 * and trajectory integration on GPU" PAPER.md:48; "local tricubics" PAPER.md:80,111; readings A27, A31 of DESIGN.md).
 * Tabulates B (direct sum O2) at s_i = i/(ngs-1), theta_j = 2 pi j/nth, zeta_k = (2 pi/nfp) k/nze (one field period)
 * on the device (the kernels run on `stream`; this is a set-up call and returns only when the table is complete, so
 * that calls on any other stream, gc_trace_host's own included, never see a half-built table), and from then on every
 * call on this field -- gc_field_eval, gc_rhs_eval, gc_trace, gc_trace_sampled, gc_trace_host, gc_trace_symplectic,
 * gc_pzeta_eval -- evaluates B and its three derivatives from a local tricubic interpolant; profiles and the
 * perturbation keep their radial tables.
 *   GC_GRID_LAGRANGE  tensor product of 4-point cubic Lagrange polynomials through the node VALUES (radial stencil
 *                     clamped as in O1, angular stencils periodic and centred on the cell); continuous, gradient jumps
 *                     at the cell faces (C0); every count >= 4; 32 ngs (nth + 3) nze bytes of device memory
 *   GC_GRID_HERMITE   tensor product of cubic Hermite polynomials through the node values AND node derivatives (f, f_s,
 *                     f_theta, f_zeta and the four mixed ones, term by term from the harmonic sum); value and gradient
 *                     continuous (C1): an adaptive integrator needs several times fewer steps on it; every count >= 2;
 *                     64 ngs (nth + 1) (nze + 1) bytes
 * Traces then run on GC_KERNEL_GRID whatever gc_set_kernel says.  (0, 0, 0) drops the grid and returns to the direct
 * sum.  The table is owned by the field.  GC_EINVAL for a count below the minimum, an unknown kind or a field with
 * kmnc / kmns -- a refused call leaves the field as it was, interpolant included; calls must not overlap traces that
 * still run on this field. */
enum { GC_GRID_LAGRANGE = 0, GC_GRID_HERMITE = 1 };
int gc_field_set_grid(gc_field* f, int32_t ngs, int32_t nth, int32_t nze, int32_t kind, void* stream);

/* O2 at n points.  DEVICE pointers.  B [n]; dB [3][n] = dB/ds, dB/dtheta, dB/dzeta, or NULL.
 * Asynchronous on `stream` (a cudaStream_t, NULL = default stream).  Used to compute mu and by tests. */
int gc_field_eval(const gc_field* f, int64_t n, const double* s, const double* th, const double* ze,
                  double* B, double* dB, void* stream);

/* The covariant radial component K at n points (NEXT-4), same layout as gc_field_eval: K [n]; dK [3][n] = dK/ds,
 * dK/dtheta, dK/dzeta, or NULL.  All zero for a field without K tables. */
int gc_kcov_eval(const gc_field* f, int64_t n, const double* s, const double* th, const double* ze,
                 double* K, double* dK, void* stream);

/* O3 at n points and time t.  DEVICE pointers.  out [9][n] = Phi, Phi_psi, Phi_theta, Phi_zeta, alpha,
 * alpha_psi, alpha_theta, alpha_zeta, alpha_t.  All zero for a static field. */
int gc_pert_eval(const gc_field* f, int64_t n, const double* s, const double* th, const double* ze,
                 double t, double* out, void* stream);

/* O4 at n states.  DEVICE pointers.  y [4][n] = s, theta, zeta, v_par (m/s); dydt [4][n] = ds/dt,
 * dtheta/dt, dzeta/dt, dv_par/dt (m/s^2).  Evaluated by the same device code path as the selected trace
 * kernel, so tests can pin the right-hand side alone. */
int gc_rhs_eval(const gc_field* f, double mass, double charge, double t, int64_t n, const double* y,
                const double* mu, double* dydt, void* stream);

/* O5-O8: trace n independent particles.  ALL ARRAY POINTERS ARE DEVICE MEMORY owned by the caller and
 * must stay valid until `stream` is synchronised; the call is asynchronous on `stream`.
 *   in : s0, th0, ze0, vpar0 (m/s), mu (J/T)         [n] each, never modified unless they alias y_out
 *        (s0 = y_out, th0 = y_out + n, ze0 = y_out + 2n, vpar0 = y_out + 3n is allowed)
 *   io : h_inout [n] or NULL: first trial step if > 0 (else params->h0); next proposal on return
 *   out: y_out [4][n] = s, theta, zeta, v_par (m/s);  t_out [n] end time (loss time when status == 1);
 *        status [n] (GC_ST_*);  n_acc, n_rej, n_forced [n] each or NULL (attempt counters);
 *        poincare [capacity][4] = particle id, t, s, theta mod 2 pi, or NULL;
 *        poincare_count: one int64 on the device, total crossings found (> capacity means the excess
 *        was dropped).  Record order is unspecified.
 * Per-particle failures are reported in `status`, never as a call failure. */
int gc_trace(const gc_field* f, const gc_trace_params* params, int64_t n,
             const double* s0, const double* th0, const double* ze0, const double* vpar0,
             const double* mu, double* h_inout,
             double* y_out, double* t_out, int32_t* status,
             int32_t* n_acc, int32_t* n_rej, int32_t* n_forced,
             double* poincare, int64_t* poincare_count, void* stream);

/* The same trace with HOST buffers.  MUTATES THE FIELD: a device workspace and a stream are created in it on the
 * first call, grown on demand and freed by gc_field_destroy, so the field is not const here and the call is not
 * re-entrant on one field: a call that overlaps another gc_trace_host call on the same field returns GC_EINVAL
 * (different fields may run concurrently).  Copies the inputs in (with GC_TRACE_RESUME also y_out, t_out, status
 * and the counters, so that untouched particles keep their values), runs gc_trace, copies every non-NULL output
 * back and synchronises.  `poincare_count` is a host int64 here.  Pinned host buffers make the copies
 * asynchronous; pageable ones work too. */
int gc_trace_host(gc_field* f, const gc_trace_params* params, int64_t n,
                  const double* s0, const double* th0, const double* ze0, const double* vpar0,
                  const double* mu, double* h_inout,
                  double* y_out, double* t_out, int32_t* status,
                  int32_t* n_acc, int32_t* n_rej, int32_t* n_forced,
                  double* poincare, int64_t* poincare_count);

/* ---- NEXT-1 of SURVEY.md section 8(f): uniform-time samples of the continuous extension and the diagnostics they
 * feed ("dense output"; "given trajectory data, transport diagnostics include ... weighted
 * Birkhoff averaging"; "the weighted Birkhoff average of P_zeta serves as an integrability
 * diagnostic, with digit accuracy below 3 indicating chaotic motion").  Readings O9, A25 of DESIGN.md section 12.
 *
 * gc_trace_sampled = gc_trace (same arguments, same results, no Poincare records) that also records the state at
 * the times tau_j = fma(j, sample_dt, sample_t0), j = 0 .. nsamp-1, from the 4th-order continuous extension of the
 * accepted step with t < tau_j <= t_new; a sample that falls on t0 is the initial state.
 *   samples    [4][nsamp][n] DEVICE: s, theta, zeta, v_par (m/s); entries not reached are left untouched
 *   sample_end [n] DEVICE int32: index of the next sample the particle would write; its valid samples are
 *              j_first <= j < sample_end with j_first = first j with tau_j >= t0 (of the first segment)
 * Under GC_TRACE_RESUME the sample grid simply continues (same sample_t0, sample_dt, buffers).  Small ensembles
 * are traced by the generic kernel (the warp kernel records no samples); GC_EINVAL if sample_dt <= 0 or a
 * buffer is NULL with nsamp > 0. */
int gc_trace_sampled(const gc_field* f, const gc_trace_params* params, int64_t n,
                     const double* s0, const double* th0, const double* ze0, const double* vpar0,
                     const double* mu, double* h_inout,
                     double* y_out, double* t_out, int32_t* status,
                     int32_t* n_acc, int32_t* n_rej, int32_t* n_forced,
                     double sample_t0, double sample_dt, int64_t nsamp, double* samples, int32_t* sample_end,
                     void* stream);

/* A17: canonical toroidal momentum P_zeta = q ((rho + alpha) G - chi(s)), rho = m v_par / (q B), at n states and
 * times.  DEVICE pointers.  y [4][n] = s, theta, zeta, v_par (m/s) (a [4][nsamp][n] sample buffer is such an array
 * with n' = nsamp n); t [n] times (alpha depends on t; may be NULL for a static field); chi_nodes [ns]: chi at the
 * radial nodes, d chi / d psi = iota, interpolated like every profile (O1); out [n] in J s / m ... (kg m^2 / s). */
int gc_pzeta_eval(const gc_field* f, double mass, double charge, int64_t n, const double* y, const double* t,
                  const double* chi_nodes, double* out, void* stream);

/* Weighted Birkhoff average of n series (A25).  DEVICE pointers.  series [nsamp][n]; for series i the samples
 * j_first <= j < (sample_end ? sample_end[i] : nsamp) are cut into two halves of N = count / 2 samples and each
 * half is averaged with the weights w_k = g((k + 1) / (N + 1)), g(x) = exp(-1 / (x (1 - x))), k = 0 .. N-1.
 * out [3][n] = WB of the first half, WB of the second half, digit accuracy
 * -log10(|WB_1 - WB_2| / max(|WB_1|, |WB_2|)) capped at 16 (NaN for series with fewer than 4 samples). */
int gc_birkhoff(int64_t n, int64_t nsamp, const double* series, int64_t j_first, const int32_t* sample_end,
                double* out, void* stream);

/* Orbit classification, characteristic frequencies and J_par of n particles from their uniform-time samples
 * ("Given trajectory data, transport diagnostics include ... characteristic orbit frequencies ... and orbit
 * classification"; reading A30 of DESIGN.md section 12).  DEVICE pointers.  samples [4][nsamp][n] as written by
 * gc_trace_sampled or gc_trace_symplectic (s, theta, zeta, v_par); the valid samples of particle i are
 * j_first <= j < (sample_end ? sample_end[i] : nsamp), taken sample_dt apart.  A reversal is a pair of consecutive
 * samples with different signs of v_par, located by the straight line through them.  out [7][n]:
 *   0 class: 0 passing (no reversal), 1 trapped;  1 number of reversals;
 *   2, 3 omega_theta, omega_zeta = (last - first angle) / elapsed time, rad/s;
 *   4 omega_bounce = 2 pi P / (time between reversal 0 and reversal 2 P), P = (reversals - 1) / 2 full periods, 0 if P = 0;
 *   5 J_par = mass * integral of v_par^2 dt over a full period (trapezoid rule, v_par = 0 at both ends), mean over the
 *     P periods, J s;  6 (max - min) / mean of it.   NaN where undefined (fewer than 2 samples; 5, 6 for P = 0). */
int gc_orbit_diagnostics(int64_t n, int64_t nsamp, const double* samples, int64_t j_first, const int32_t* sample_end,
                         double sample_dt, double mass, double* out, void* stream);

/* ---- NEXT-3 of SURVEY.md section 8(f): the symplectic integrator ("A symplectic integrator for
 * non-canonical guiding-center orbits uses the explicit-implicit Euler scheme of (Albert et al., 2020)"; PAPER.md:60-62,
 * Fig. 1 left: "the symplectic algorithm exhibits a stable moving time average of the energy").  Reading A28 of
 * static fields with K = 0 (GC_EINVAL for a field with modes or kmnc / kmns); canonical momenta
 * p_theta = q (psi0 s + rho I), p_zeta = q (rho G - chi), rho = m v_par / (q B); state (s, theta, zeta, p_zeta); one
 * step of size dt solves  p_theta' - p_theta + dt dH/dtheta = 0,  p_zeta' - p_zeta + dt dH/dzeta = 0  for
 * (s', p_zeta') at the old angles (to a last update below newton_tol max(1, |x|) of x = (s, p_zeta / (q psi0)),
 * status 4 after max_iter iterations) and then advances the angles explicitly with the derivatives of H at the new
 * (s', p_zeta').  Works on the direct harmonic sum (ensembles of at least GC_TILE_MIN_PARTICLES on the cell-binned mma
 * engine, one pass per field evaluation; smaller ones, sampled ones and GC_KERNEL_GENERIC on the lane kernel) and on
 * the 3-D interpolants of gc_field_set_grid.
 * The 2 x 2 system is solved by a quasi-Newton iteration that keeps the Jacobian of the dt = 0 part of the equations
 * (one field evaluation per iteration, started from the linear extrapolation of the last step).  It contracts like
 * dt times the gradient scale of H: for steps well below the bounce and drift times -- the regime of the method, a few
 * percent of a transit time, where it takes 4 to 6 iterations -- it reaches newton_tol; for a dt of the order of the
 * transit time it does not converge where a full Newton iteration still would, and the particle ends with status
 * GC_ST_NONFINITE after max_iter iterations.  Reduce dt then; raising max_iter does not help. */
typedef struct {
  double mass, charge;        /* kg, C                                                              */
  double t0, dt;              /* s; fixed step dt > 0                                               */
  int64_t nsteps;             /* steps per particle and call                                        */
  double s_loss, s_min;       /* stop rules of O7, checked after every step                         */
  double newton_tol;          /* e.g. 1e-13                                                         */
  int64_t max_iter;           /* e.g. 50                                                            */
  int64_t flags;              /* 0 or GC_TRACE_RESUME (skip particles whose status is not 0; counters add up) */
} gc_symplectic_params;

/* DEVICE pointers, asynchronous on `stream`.
 *   in : s0, th0, ze0, vpar0 (m/s), mu (J/T) [n] (may alias the rows of y_out as in gc_trace);
 *        chi_nodes [ns]: chi at the radial nodes, d chi / d psi = iota, interpolated like every profile (O1); the
 *        integrator takes d chi / d s from THAT interpolant where the equations of motion have psi0 iota
 *   out: y_out [4][n] = s, theta, zeta, v_par (m/s); t_out [n] = t0 + steps dt; status [n]: GC_ST_TMAX (all steps
 *        done), GC_ST_LOST, GC_ST_AXIS, GC_ST_NONFINITE (iteration failed or a non-finite value: the state before
 *        the failed step is reported); n_steps, n_iter [n] or NULL: steps taken, iterations in total
 *   samples [4][nsamp][n] or nsamp = 0: sample 0 = the initial state, sample j = the state after step
 *        j * sample_stride; sample_end [n] = samples written (under GC_TRACE_RESUME the count continues from
 *        sample_end; nsteps should then be a multiple of sample_stride). */
int gc_trace_symplectic(const gc_field* f, const gc_symplectic_params* params, int64_t n,
                        const double* s0, const double* th0, const double* ze0, const double* vpar0,
                        const double* mu, const double* chi_nodes,
                        double* y_out, double* t_out, int32_t* status, int32_t* n_steps, int32_t* n_iter,
                        int64_t sample_stride, int64_t nsamp, double* samples, int32_t* sample_end, void* stream);

/* Kernel choice (GC_KERNEL_*) for later gc_trace / gc_rhs_eval calls on this field (default AUTO); GC_EINVAL
 * if the field does not fit the requested kernel. */
int gc_set_kernel(gc_field* f, int32_t kernel);
/* Tuning of the cell-binned kernels (MMA, TILE) for later calls on this field; results do not depend on either.
 *   GC_OPT_WAVE_PARTICLES  number of record slots: a larger ensemble streams through them inside one launch (a
 *                          finished particle hands its slot to the next unstarted one), so that the per-particle
 *                          records (128 B each) stay in L2 between epochs; 0 = automatic (2^18), minimum 4096; an
 *                          ensemble up to 1.25 times this number gets one slot per particle
 *   GC_OPT_CHUNK_ATTEMPTS  attempted steps a particle gets per epoch before the ensemble is re-binned by radial
 *                          cell; 0 = the kernel's default (8), at most the kernel's compiled maximum (8)
 * GC_EINVAL for an unknown option or a value out of range. */
enum { GC_OPT_WAVE_PARTICLES = 1, GC_OPT_CHUNK_ATTEMPTS = 2 };
int gc_set_option(gc_field* f, int32_t option, int64_t value);
/* Which kernel gc_trace will launch for this field and n particles (GC_KERNEL_GENERIC, _WARP, _TILE or _MMA), and
 * its launch geometry; any pointer may be NULL. */
int gc_kernel_info(const gc_field* f, int64_t n, int32_t* kernel, int32_t* blocks, int32_t* threads_per_block,
                   int32_t* smem_bytes, int32_t* regs_per_thread);

/* ---- gc_trace for callers that must not allocate device memory.
 *
 * Who needs it.  gc_trace borrows its per-call work area (one 128-byte record per particle plus the index arrays of the
 * cell binning) from a stream-ordered memory pool, and the first call of a given size makes that pool ask the driver for
 * memory.  Some programs that embed this library cannot afford that once they are up: a long-running service that gave
 * the whole GPU to its own arena at start-up and treats every later driver allocation as a budget violation (or simply
 * has none left to give); a control or acquisition loop with a deadline, for which the unbounded latency and the
 * device-wide synchronisation an allocation or a release can cause are not acceptable; a plug-in whose host forbids the
 * CUDA allocation calls outside its own allocator.  For them gc_trace_noalloc traces with the work area in a fixed
 * array that is part of the library image: GC_NOALLOC_SCRATCH_BYTES (5 MiB) of device memory on every GPU that loads
 * libgcorbit.so, held until the process exits whether or not this function is ever called.
 *
 * What it does.  The arguments, the results and the asynchronous behaviour on `stream` are those of gc_trace with
 * GC_KERNEL_MMA selected (same kernel, same launch geometry; only the address of the work area differs).  It never
 * calls cudaMalloc, cudaFree, their stream-ordered forms or any library routine that allocates; inputs and outputs
 * remain the caller's device buffers.
 *
 * Limits.  n <= GC_NOALLOC_MAX_PARTICLES (32768; one record slot per particle) and the binning arrays of the field must
 * fit the rest of the array (they do up to several thousand radial nodes): beyond either the call returns GC_EINVAL and
 * gc_last_error() says which limit and by how much -- trace a larger ensemble as consecutive slices.  The field must fit
 * the mma kernel (max |xn| <= 16, max xm <= 16) and must not have a 3-D interpolant set; GC_EINVAL otherwise.
 *
 * Set-up.  The first call on each GPU looks up the device address of the array (one cudaGetSymbolAddress, with that
 * GPU current) and remembers it; make that first call during start-up, before any stream capture.  Call with the
 * field's GPU current, as for every other entry point.
 *
 * Sharing.  There is ONE array per GPU and every call uses it.  A call clears the counters it needs at zero itself (in
 * stream order), so what the previous call left behind never matters; but two calls that can run on the GPU at the same
 * time -- different streams, or different host threads on different streams, also through different fields -- would
 * overwrite each other's records and return garbage.  Issue all gc_trace_noalloc calls on one stream, or order them
 * with events.  gc_trace itself is not affected and may run next to it. */
enum { GC_NOALLOC_MAX_PARTICLES = 32768, GC_NOALLOC_SCRATCH_BYTES = 5 * 1024 * 1024 };
int gc_trace_noalloc(const gc_field* f, const gc_trace_params* params, int64_t n,
                     const double* s0, const double* th0, const double* ze0, const double* vpar0,
                     const double* mu, double* h_inout,
                     double* y_out, double* t_out, int32_t* status,
                     int32_t* n_acc, int32_t* n_rej, int32_t* n_forced,
                     double* poincare, int64_t* poincare_count, void* stream);

/* Thread-local text of the last nonzero return ("" if none). */
const char* gc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
