/* gc_oracle.h -- CPU ORACLE for the guiding-centre hot path.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision restatement of what the path computes, written from the paper
 * (/root/reference/PAPER.md at survey time; cited below as PAPER.md:<line>) and, where the paper prints
 * no mathematics, from the readings O1-O8 / A1-A22 recorded in SURVEY.md section 8(c) and DESIGN.md.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
 * this library.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_2605_16734_b200/csrc/ and include/.
 *
 * Pins (tests/test_oracle_*.py): Lagrange weights vs polynomial exactness and scipy; harmonic sums vs
 * finite differences and an independent numpy series; DP5 tableau vs exact-rational order conditions
 * and scipy's RK45 step; the RHS vs the Euler-Lagrange equations of the guiding-centre Lagrangian
 * solved numerically; energy, P_zeta, helical momentum, n*H - omega*P_zeta invariants; closed-form
 * orbits; brute-force RK4; (tests/test_oracle_sampling.py) uniform-time samples vs closed form and an independent
 * DOP853 integration, P_zeta of the samples vs conservation laws, the weighted Birkhoff average (oracle/__init__.py)
 * vs super-convergence on quasi-periodic signals and the logistic map.  FIRM3D-level agreement (same numbers as the reference code on its own
 * equilibria) is PARITY UNPINNED: no code, equilibrium file or printed equation exists to pin it to.
 */
#ifndef GC_ORACLE_H
#define GC_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Field description: harmonics on a uniform radial grid s_j = j/(ns-1). Host pointers,
 * copied by oracle_field_create. */
typedef struct {
  int32_t ns, nfp, nh;
  const int32_t *xm, *xn;      /* [nh]; phase m*theta - n*nfp*zeta                         */
  const double *bmnc;          /* [ns][nh] node-major                                      */
  const double *G, *I, *iota;  /* [ns]                                                     */
  double psi0;                 /* psi = psi0 * s                                           */
  int32_t nk;                  /* perturbation harmonics, 0 = static                       */
  const int32_t *mode_m, *mode_n;          /* [nk]; phase m*theta - n*zeta + omega*t + phase */
  const double *mode_omega, *mode_phase;   /* [nk]                                          */
  const double *phihat;        /* [ns][nk] node-major, volts                               */
  /* NEXT-4 of SURVEY.md section 8(f) (field model of PAPER.md:44 without stellarator symmetry and with the covariant
   * radial component kept); each may be NULL (= zero): */
  const double *bmns;          /* [ns][nh] sin coefficients of B:  B += bmns sin(m theta - n nfp zeta)            */
  const double *kmnc, *kmns;   /* [ns][nh] covariant radial component K (B = G grad zeta + I grad theta + K grad psi),
                                  T/m ... in units of T m / (T m^2) = 1/m: K = sum kmnc cos + kmns sin            */
} oracle_field_desc;

typedef struct oracle_field oracle_field;

typedef struct {
  double mass, charge;
  double t0, t_max;
  double rtol, atol;
  double v_ref;
  double h0, h_min;
  double s_loss, s_min;
  int64_t max_steps;
  int64_t poincare_capacity;   /* records in the shared buffer; 0 disables O8 */
  int64_t traj_capacity;       /* per-particle accepted-step records; 0 disables (oracle-only) */
  int64_t section;             /* which crossings the Poincare records hold: 0 zeta = 0 mod 2 pi (O8), 1 v_par = 0 (O8b) */
  int64_t refine_loss;         /* O7b: 1 = a lost particle reports the root of s(tau) = s_loss on the continuous
                                  extension of its last step (t_out, y_out) instead of the end of that step (A8) */
} oracle_trace_params;

oracle_field *oracle_field_create(const oracle_field_desc *d);
void oracle_field_destroy(oracle_field *f);

/* O1: stencil start i0, x = s*(ns-1) - i0, cubic Lagrange weights w[4] and d/ds weights dw[4]. */
void oracle_lagrange(int32_t ns, double s, int32_t *i0, double w[4], double dw[4]);

/* O2: out = {B, dB/ds, dB/dtheta, dB/dzeta}. */
void oracle_eval_B(const oracle_field *f, double s, double th, double ze, double out[4]);
/* The direct sum O2 whatever oracle_field_set_grid says. */
void oracle_eval_B_sum(const oracle_field *f, double s, double th, double ze, double out[4]);
/* NEXT-2 (reading A27): replace the direct sum by a local tricubic interpolant.
 * oracle_field_set_grid tabulates B (direct sum O2) at s_i = i/(ngs-1), theta_j = 2 pi j/nth,
 * zeta_k = (2 pi/nfp) k/nze (each count >= 4; 0,0,0 switches back to the direct sum) and from then on oracle_eval_B,
 * and with it oracle_rhs, oracle_trace and oracle_pzeta, evaluate B and its three derivatives as the tensor-product
 * cubic Lagrange interpolant of those node values (radial stencil as O1, angular stencils periodic and centred).
 * Fields with K tables are rejected by the CUDA path; the oracle interpolates B only.  Returns 0, -1 on bad sizes. */
int oracle_field_set_grid(oracle_field *f, int32_t ngs, int32_t nth, int32_t nze);
const double *oracle_field_grid(const oracle_field *f);           /* [ngs][nth][nze] or NULL */
void oracle_eval_B_grid(const oracle_field *f, double s, double th, double ze, double out[4]);
/* NEXT-2, second reading (A31): the C1 tricubic Hermite interpolant.  oracle_field_set_grid_hermite tabulates B and
 * its seven first and mixed derivatives (f, f_s, f_th, f_ze, f_s_th, f_s_ze, f_th_ze, f_s_th_ze; direct sum, term by
 * term) on the same node grid (each count >= 2; 0,0,0 switches back) and from then on oracle_eval_B evaluates the
 * tensor-product cubic Hermite interpolant of the cell that holds the point.  Drops a Lagrange grid and vice versa. */
int oracle_field_set_grid_hermite(oracle_field *f, int32_t ngs, int32_t nth, int32_t nze);
const double *oracle_field_grid8(const oracle_field *f);          /* [ngs][nth][nze][8] or NULL */
void oracle_eval_B_hermite(const oracle_field *f, double s, double th, double ze, double out[4]);
/* The direct sum with its mixed derivatives: out = {f, f_s, f_th, f_ze, f_s_th, f_s_ze, f_th_ze, f_s_th_ze}. */
void oracle_eval_B_mixed(const oracle_field *f, double s, double th, double ze, double out[8]);
/* NEXT-4: covariant radial component, out = {K, dK/ds, dK/dtheta, dK/dzeta} (all zero without K tables). */
void oracle_eval_K(const oracle_field *f, double s, double th, double ze, double out[4]);
/* O1 on profiles: out = {G, dG/ds, I, dI/ds, iota, diota/ds}. */
void oracle_eval_profiles(const oracle_field *f, double s, double out[6]);
/* O3: out = {Phi, Phi_psi, Phi_theta, Phi_zeta, alpha, alpha_psi, alpha_theta, alpha_zeta, alpha_t}. */
void oracle_eval_pert(const oracle_field *f, double s, double th, double ze, double t, double out[9]);

/* O4: y = (s, theta, zeta, u = v_par/v_ref); dydt likewise. */
void oracle_rhs(const oracle_field *f, double mass, double charge, double mu, double v_ref,
                double t, const double y[4], double dydt[4]);

/* O4 in its general form (NEXT-4): the Euler-Lagrange equations of
 *   L = q rho_c K psidot + q (psi + rho_c I) thetadot + q (rho_c G - chi) zetadot - H
 * written as the 4 x 4 antisymmetric system  sum_j omega_ij zdot_j = dH/dz_i + q dA*_i/dt  (z = psi, theta, zeta,
 * v_par) and solved by Gaussian elimination.  oracle_rhs uses this form whenever the field has K tables; for K = 0
 * it equals the closed form of oracle_rhs (pinned). */
void oracle_rhs_general(const oracle_field *f, double mass, double charge, double mu, double v_ref,
                        double t, const double y[4], double dydt[4]);

/* O5: one Dormand-Prince attempt of size h from (t, y) with k1 = f(t, y) given.
 * Outputs y_new (5th order), k[7][4] (k[0] = k1 copied, k[6] = f(t+h, y_new)), delta[4] (embedded error). */
void oracle_dp5_attempt(const oracle_field *f, double mass, double charge, double mu, double v_ref,
                        double t, const double y[4], const double k1[4], double h,
                        double y_new[4], double k[7][4], double delta[4]);
/* The same attempt on an arbitrary 4-component right-hand side (used by the tableau pins). */
typedef void (*oracle_rhs_fn)(void *ctx, double t, const double y[4], double dydt[4]);
void oracle_dp5_attempt_fn(oracle_rhs_fn fn, void *ctx, double t, const double y[4], const double k1[4],
                           double h, double y_new[4], double k[7][4], double delta[4]);
/* O8: continuous extension at t + tau*h, tau in [0,1]. */
void oracle_dp5_dense(const double y[4], const double y_new[4], const double k[7][4], double h,
                      double tau, double y_tau[4]);
/* O6: error norm and the two step-size factors. */
double oracle_err_norm(const double y[4], const double y_new[4], const double delta[4],
                       double rtol, double atol);
double oracle_scale_accept(double err);   /* factor applied to h after an accepted attempt */
double oracle_scale_reject(double err);   /* factor applied to h after a rejected attempt  */

/* O5-O8: trace n particles (OpenMP over particles only).  All arrays host memory.
 * y_out [4][n]; status 0 t_max, 1 lost, 2 axis, 3 max_steps, 4 non-finite/stalled.
 * traj [n][traj_capacity][5] = (t, s, theta, zeta, u) after each accepted step (oracle-only diagnostic).
 * poincare [cap][4] = (id, t, s, theta mod 2pi); *poincare_count counts all hits (may exceed cap).
 * Returns 0, or -1 on bad arguments. */
int oracle_trace(const oracle_field *f, const oracle_trace_params *p, int64_t n,
                 const double *s0, const double *th0, const double *ze0, const double *vpar0,
                 const double *mu, double *h_inout,
                 double *y_out, double *t_out, int32_t *status,
                 int32_t *n_acc, int32_t *n_rej, int32_t *n_forced,
                 double *poincare, int64_t *poincare_count,
                 double *traj, int64_t *traj_count);

/* O9 (NEXT-1 of SURVEY.md section 8(f); "dense output", "given trajectory data, transport
 * diagnostics include ... weighted Birkhoff averaging"): the same trace, recording the state at the uniform times
 * tau_j = sample_t0 + j sample_dt, j = 0 .. nsamp-1, from the continuous extension of the accepted step that
 * contains tau_j (t < tau_j <= t_new; a sample that falls on t0 is the initial state).
 * samples [4][nsamp][n] = s, theta, zeta, v_par (m/s); sample_end [n] = index of the next sample the particle
 * would have written: its samples j_first <= j < sample_end are valid, j_first = first j with tau_j >= t0; a
 * particle that stops early leaves the later ones untouched. */
int oracle_trace_sampled(const oracle_field *f, const oracle_trace_params *p, int64_t n,
                         const double *s0, const double *th0, const double *ze0, const double *vpar0,
                         const double *mu, double *h_inout,
                         double *y_out, double *t_out, int32_t *status,
                         int32_t *n_acc, int32_t *n_rej, int32_t *n_forced,
                         double sample_t0, double sample_dt, int64_t nsamp, double *samples, int32_t *sample_end);

/* A17: P_zeta = q ((rho + alpha) G - chi), rho = m v_par / (q B); chi_nodes [ns] = chi at the radial nodes. */
double oracle_pzeta(const oracle_field *f, double mass, double charge, const double *chi_nodes,
                    double s, double th, double ze, double vpar, double t);

/* ---- NEXT-3: the symplectic explicit-implicit Euler integrator for static fields
 * with K = 0 (reading A28; the scheme is written out above oracle_symplectic_step in gc_oracle.c).  State
 * z = (s, theta, zeta, p_zeta); chi_nodes [ns] = chi at the radial nodes (d chi / d psi = iota), interpolated by O1. */
typedef struct {
  double mass, charge;
  double t0, dt;               /* fixed step, s                                             */
  int64_t nsteps;              /* steps per particle                                        */
  double s_loss, s_min;        /* stop rules of O7                                          */
  double newton_tol;           /* relative size of the last Newton update, e.g. 1e-13       */
} oracle_symplectic_params;

/* One step of size h on z = (s, theta, zeta, p_zeta); returns 0, -1 if Newton did not converge. */
int oracle_symplectic_step(const oracle_field *f, double mass, double charge, double mu, const double *chi_nodes,
                           double h, double newton_tol, double z[4], int32_t *iterations);
double oracle_symplectic_pzeta(const oracle_field *f, double mass, double charge, const double *chi_nodes,
                               double s, double th, double ze, double vpar);
double oracle_symplectic_vpar(const oracle_field *f, double mass, double charge, const double *chi_nodes,
                              double s, double th, double ze, double pz);
/* n particles, nsteps steps each (OpenMP over particles).  y_out [4][n] = s, theta, zeta, v_par (m/s); t_out [n];
 * status 0 all steps done, 1 lost, 2 axis, 4 Newton failure / non-finite; n_steps, n_iter [n] or NULL (steps taken,
 * Newton iterations in total).  samples [4][nsamp][n] (or nsamp = 0): sample 0 = the initial state, sample j = the
 * state after step j * sample_stride; sample_end [n] = samples written.  Returns 0, -1 on bad arguments (among them:
 * a field with modes or K tables). */
int oracle_trace_symplectic(const oracle_field *f, const oracle_symplectic_params *p, int64_t n,
                            const double *s0, const double *th0, const double *ze0, const double *vpar0,
                            const double *mu, const double *chi_nodes,
                            double *y_out, double *t_out, int32_t *status, int32_t *n_steps, int32_t *n_iter,
                            int64_t sample_stride, int64_t nsamp, double *samples, int32_t *sample_end);

/* Check (d): classical fixed-step RK4, nsteps steps of size h from t0; y_out [4][n]. */
void oracle_rk4(const oracle_field *f, double mass, double charge, double v_ref, int64_t n,
                const double *s0, const double *th0, const double *ze0, const double *vpar0,
                const double *mu, double t0, double h, int64_t nsteps, double *y_out);

int oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
