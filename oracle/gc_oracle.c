/* gc_oracle.c -- CPU ORACLE (test infrastructure, not the product).  See gc_oracle.h.
 *
 * Plain C, FP64, one libm sin + cos per harmonic, sequential sums in index order, no blocking, no
 * fusion, no reordering: written so that each function can be checked against the cited passage by
 * eye.  OpenMP is used over particles only ("trajectories are independent").
 */
#include "gc_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

struct oracle_field {
  int32_t ns, nfp, nh, nk;
  int32_t *xm, *xn, *mode_m, *mode_n;
  double *bmnc, *G, *I, *iota, *mode_omega, *mode_phase, *phihat;
  double *bmns, *kmnc, *kmns;          /* NEXT-4: NULL = absent */
  double psi0;
  /* NEXT-2: node values of B on the (s, theta, zeta) grid, [ngs][nth][nze]; NULL = the direct harmonic sum */
  int32_t ngs, nth, nze;
  double *grid;
  /* the Hermite variant (reading A31): per node the 8 values f, f_s, f_th, f_ze, f_s_th, f_s_ze, f_th_ze, f_s_th_ze,
     [ngs][nth][nze][8]; NULL unless oracle_field_set_grid_hermite was called */
  double *grid8;
};

static void *dup_mem(const void *src, size_t bytes) {
  void *p = malloc(bytes ? bytes : 1);
  if (p && bytes) memcpy(p, src, bytes);
  return p;
}

oracle_field *oracle_field_create(const oracle_field_desc *d) {
  if (!d || d->ns < 4 || d->nh < 1 || d->nk < 0) return NULL;
  oracle_field *f = (oracle_field *)calloc(1, sizeof(*f));
  f->ns = d->ns; f->nfp = d->nfp; f->nh = d->nh; f->nk = d->nk; f->psi0 = d->psi0;
  f->xm = (int32_t *)dup_mem(d->xm, sizeof(int32_t) * d->nh);
  f->xn = (int32_t *)dup_mem(d->xn, sizeof(int32_t) * d->nh);
  f->bmnc = (double *)dup_mem(d->bmnc, sizeof(double) * (size_t)d->ns * d->nh);
  f->G = (double *)dup_mem(d->G, sizeof(double) * d->ns);
  f->I = (double *)dup_mem(d->I, sizeof(double) * d->ns);
  f->iota = (double *)dup_mem(d->iota, sizeof(double) * d->ns);
  if (d->nk > 0) {
    f->mode_m = (int32_t *)dup_mem(d->mode_m, sizeof(int32_t) * d->nk);
    f->mode_n = (int32_t *)dup_mem(d->mode_n, sizeof(int32_t) * d->nk);
    f->mode_omega = (double *)dup_mem(d->mode_omega, sizeof(double) * d->nk);
    f->mode_phase = (double *)dup_mem(d->mode_phase, sizeof(double) * d->nk);
    f->phihat = (double *)dup_mem(d->phihat, sizeof(double) * (size_t)d->ns * d->nk);
  }
  size_t tab = sizeof(double) * (size_t)d->ns * d->nh;
  if (d->bmns) f->bmns = (double *)dup_mem(d->bmns, tab);
  if (d->kmnc) f->kmnc = (double *)dup_mem(d->kmnc, tab);
  if (d->kmns) f->kmns = (double *)dup_mem(d->kmns, tab);
  return f;
}

void oracle_field_destroy(oracle_field *f) {
  if (!f) return;
  free(f->xm); free(f->xn); free(f->bmnc); free(f->G); free(f->I); free(f->iota);
  free(f->mode_m); free(f->mode_n); free(f->mode_omega); free(f->mode_phase); free(f->phihat);
  free(f->bmns); free(f->kmnc); free(f->kmns); free(f->grid); free(f->grid8);
  free(f);
}

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ---- O1: radial cubic Lagrange interpolation on the uniform grid -------------------- */
void oracle_lagrange(int32_t ns, double s, int32_t *i0_out, double w[4], double dw[4]) {
  double u = s * (double)(ns - 1);
  double c = floor(u);
  int32_t i0;
  if (!(c >= 1.0)) i0 = 0;                         /* also catches NaN */
  else if (c - 1.0 >= (double)(ns - 4)) i0 = ns - 4;
  else i0 = (int32_t)c - 1;
  double x = u - (double)i0;                       /* nodes of the stencil sit at x = 0,1,2,3 */
  w[0] = -(x - 1.0) * (x - 2.0) * (x - 3.0) / 6.0;
  w[1] = x * (x - 2.0) * (x - 3.0) / 2.0;
  w[2] = -x * (x - 1.0) * (x - 3.0) / 2.0;
  w[3] = x * (x - 1.0) * (x - 2.0) / 6.0;
  double scale = (double)(ns - 1);                 /* d/ds = (ns-1) d/dx */
  dw[0] = -((x - 2.0) * (x - 3.0) + (x - 1.0) * (x - 3.0) + (x - 1.0) * (x - 2.0)) / 6.0 * scale;
  dw[1] = ((x - 2.0) * (x - 3.0) + x * (x - 3.0) + x * (x - 2.0)) / 2.0 * scale;
  dw[2] = -((x - 1.0) * (x - 3.0) + x * (x - 3.0) + x * (x - 1.0)) / 2.0 * scale;
  dw[3] = ((x - 1.0) * (x - 2.0) + x * (x - 2.0) + x * (x - 1.0)) / 6.0 * scale;
  *i0_out = i0;
}

/* value and d/ds of one tabulated quantity with row stride `stride` */
static void interp(const double *tab, int32_t stride, int32_t i0, const double w[4], const double dw[4],
                   double *val, double *dval) {
  double v = 0.0, d = 0.0;
  for (int j = 0; j < 4; ++j) {
    double t = tab[(size_t)(i0 + j) * stride];
    v += w[j] * t;
    d += dw[j] * t;
  }
  *val = v; *dval = d;
}

/* ---- O2: equilibrium field strength and its derivatives -------------------------------------------
 * One Fourier series  X = sum_k [ xc_k(s) cos(ang_k) + xs_k(s) sin(ang_k) ],  ang_k = m_k theta - n_k nfp zeta, and
 * its derivatives in s, theta, zeta; either table may be NULL.  One libm cos + sin per harmonic, index order. */
static void eval_series(const oracle_field *f, const double *tabc, const double *tabs,
                        double s, double th, double ze, double out[4]) {
  int32_t i0; double w[4], dw[4];
  oracle_lagrange(f->ns, s, &i0, w, dw);
  double X = 0.0, Xs = 0.0, Xth = 0.0, Xze = 0.0;
  for (int k = 0; k < f->nh; ++k) {
    double m = (double)f->xm[k], nn = (double)f->xn[k] * (double)f->nfp;
    double ang = m * th - nn * ze;
    double c = cos(ang), sn = sin(ang);
    if (tabc) {
      double b, bs;
      interp(tabc + k, f->nh, i0, w, dw, &b, &bs);
      X += b * c;
      Xs += bs * c;
      Xth += -m * b * sn;
      Xze += nn * b * sn;
    }
    if (tabs) {                                    /* NEXT-4: the terms stellarator symmetry forbids */
      double b, bs;
      interp(tabs + k, f->nh, i0, w, dw, &b, &bs);
      X += b * sn;
      Xs += bs * sn;
      Xth += m * b * c;
      Xze += -nn * b * c;
    }
  }
  out[0] = X; out[1] = Xs; out[2] = Xth; out[3] = Xze;
}

void oracle_eval_B_sum(const oracle_field *f, double s, double th, double ze, double out[4]) {
  eval_series(f, f->bmnc, f->bmns, s, th, ze, out);
}

/* ---- NEXT-2 ("CUDA kernels implement field interpolation", "local
 * tricubics"; reading A27 of DESIGN.md): B as a local tricubic interpolant of its own node values.
 * Grid: s_i = i/(ngs-1), theta_j = 2 pi j/nth, zeta_k = (2 pi/nfp) k/nze (one field period; both angles periodic).
 * Node values come from the direct sum O2.  Evaluation: tensor product of the cubic Lagrange weights of O1 in each
 * direction; the radial stencil is clamped as in O1, an angular stencil is the four nodes c-1 .. c+2 around the
 * cell c = floor(u), u = angle * (nodes per radian), taken modulo the period. */
static const double ORACLE_TWO_PI = 6.283185307179586476925286766559;

int oracle_field_set_grid(oracle_field *f, int32_t ngs, int32_t nth, int32_t nze) {
  if (!f) return -1;
  free(f->grid); f->grid = NULL; f->ngs = f->nth = f->nze = 0;
  free(f->grid8); f->grid8 = NULL;
  if (ngs == 0 && nth == 0 && nze == 0) return 0;                 /* back to the direct sum */
  if (ngs < 4 || nth < 4 || nze < 4) return -1;
  double *g = (double *)malloc(sizeof(double) * (size_t)ngs * nth * nze);
  if (!g) return -1;
#pragma omp parallel for collapse(2) schedule(static)
  for (int i = 0; i < ngs; ++i)
    for (int j = 0; j < nth; ++j)
      for (int k = 0; k < nze; ++k) {
        double s = (double)i / (double)(ngs - 1);
        double th = ORACLE_TWO_PI * (double)j / (double)nth;
        double ze = ORACLE_TWO_PI * (double)k / ((double)nze * (double)f->nfp);
        double out[4];
        oracle_eval_B_sum(f, s, th, ze, out);
        g[((size_t)i * nth + j) * nze + k] = out[0];
      }
  f->grid = g; f->ngs = ngs; f->nth = nth; f->nze = nze;
  return 0;
}

const double *oracle_field_grid(const oracle_field *f) { return f->grid; }

/* cubic Lagrange weights on a periodic uniform grid of `nodes` points per `period`: first node j0 (before the
 * modulo), weights w[4], d/d(angle) weights dw[4].  x = u - j0 lies in [1, 2): the stencil is always centred. */
static void periodic_weights(int32_t nodes, double nodes_per_radian, double angle, int64_t *j0_out,
                             double w[4], double dw[4]) {
  double u = angle * nodes_per_radian;
  double c = floor(u);
  double x = u - (c - 1.0);
  w[0] = -(x - 1.0) * (x - 2.0) * (x - 3.0) / 6.0;
  w[1] = x * (x - 2.0) * (x - 3.0) / 2.0;
  w[2] = -x * (x - 1.0) * (x - 3.0) / 2.0;
  w[3] = x * (x - 1.0) * (x - 2.0) / 6.0;
  dw[0] = -((x - 2.0) * (x - 3.0) + (x - 1.0) * (x - 3.0) + (x - 1.0) * (x - 2.0)) / 6.0 * nodes_per_radian;
  dw[1] = ((x - 2.0) * (x - 3.0) + x * (x - 3.0) + x * (x - 2.0)) / 2.0 * nodes_per_radian;
  dw[2] = -((x - 1.0) * (x - 3.0) + x * (x - 3.0) + x * (x - 1.0)) / 2.0 * nodes_per_radian;
  dw[3] = ((x - 1.0) * (x - 2.0) + x * (x - 2.0) + x * (x - 1.0)) / 6.0 * nodes_per_radian;
  double r = fmod(c - 1.0, (double)nodes);           /* exact: both are integers below 2^53 */
  if (r < 0.0) r += (double)nodes;
  *j0_out = (int64_t)r;
}

void oracle_eval_B_grid(const oracle_field *f, double s, double th, double ze, double out[4]) {
  int32_t i0; double ws[4], dws[4], wt[4], dwt[4], wz[4], dwz[4];
  int64_t j0, k0;
  oracle_lagrange(f->ngs, s, &i0, ws, dws);
  periodic_weights(f->nth, (double)f->nth / ORACLE_TWO_PI, th, &j0, wt, dwt);
  periodic_weights(f->nze, (double)f->nze * (double)f->nfp / ORACLE_TWO_PI, ze, &k0, wz, dwz);
  double B = 0.0, Bs = 0.0, Bt = 0.0, Bz = 0.0;
  for (int a = 0; a < 4; ++a)
    for (int b = 0; b < 4; ++b)
      for (int c = 0; c < 4; ++c) {
        int64_t j = (j0 + b) % f->nth, k = (k0 + c) % f->nze;
        double v = f->grid[((size_t)(i0 + a) * f->nth + j) * f->nze + k];
        B += ws[a] * wt[b] * wz[c] * v;
        Bs += dws[a] * wt[b] * wz[c] * v;
        Bt += ws[a] * dwt[b] * wz[c] * v;
        Bz += ws[a] * wt[b] * dwz[c] * v;
      }
  out[0] = B; out[1] = Bs; out[2] = Bt; out[3] = Bz;
}

/* ---- NEXT-2, second reading (A31 of DESIGN.md): "local tricubics" as the C1 tricubic HERMITE
 * interpolant.  Every node carries the value of B and its seven first and mixed derivatives
 *     f, f_s, f_th, f_ze, f_s_th, f_s_ze, f_th_ze, f_s_th_ze
 * (direct sum O2 and its term-by-term derivatives; the s-derivatives are those of the radial Lagrange interpolant of
 * O1 on the stencil that O1 picks AT the node).  In the cell [s_i, s_i+1] x [th_j, th_j+1] x [ze_k, ze_k+1] with
 * local coordinates x, y, z in [0, 1) the interpolant is the tensor product of the 1-D cubic Hermite basis
 *     h00 = 1 - 3x^2 + 2x^3 (value at 0)   h10 = 3x^2 - 2x^3 (value at 1)
 *     h01 = x - 2x^2 + x^3  (slope at 0)   h11 = -x^2 + x^3  (slope at 1)        slopes scaled by the cell width:
 *     f = sum over corners (a, b, c) and derivative orders (p, q, r) in {0,1}^3 of
 *         D[corner][p q r] (ds)^p (dth)^q (dze)^r  h_{a p}(x) h_{b q}(y) h_{c r}(z)
 * and its derivatives are the derivatives of that polynomial.  Value and gradient are continuous across cell faces
 * (C1), unlike the Lagrange variant above.  Radial cell: i = clamp(floor(s (ngs-1)), 0, ngs-2) (extrapolates outside
 * [0, 1] like O1); angular cells periodic. */
static void eval_series_mixed(const oracle_field *f, double s, double th, double ze, double out[8]) {
  int32_t i0; double w[4], dw[4];
  oracle_lagrange(f->ns, s, &i0, w, dw);
  for (int q = 0; q < 8; ++q) out[q] = 0.0;
  for (int k = 0; k < f->nh; ++k) {
    double m = (double)f->xm[k], nn = (double)f->xn[k] * (double)f->nfp;
    double ang = m * th - nn * ze;
    double c = cos(ang), sn = sin(ang);
    for (int pass = 0; pass < 2; ++pass) {
      const double *tab = pass == 0 ? f->bmnc : f->bmns;
      if (!tab) continue;
      double b, bs;
      interp(tab + k, f->nh, i0, w, dw, &b, &bs);
      /* pass 0: b cos(ang); pass 1: b sin(ang).  d/dth: -m sin | m cos; d/dze: nn sin | -nn cos;
         d2/dth dze: m nn cos | m nn sin */
      double v = pass == 0 ? c : sn;
      double vth = pass == 0 ? -m * sn : m * c;
      double vze = pass == 0 ? nn * sn : -nn * c;
      double vtz = pass == 0 ? m * nn * c : m * nn * sn;
      out[0] += b * v;   out[1] += bs * v;
      out[2] += b * vth; out[3] += b * vze;
      out[4] += bs * vth; out[5] += bs * vze;
      out[6] += b * vtz; out[7] += bs * vtz;
    }
  }
}

void oracle_eval_B_mixed(const oracle_field *f, double s, double th, double ze, double out[8]) {
  eval_series_mixed(f, s, th, ze, out);
}

int oracle_field_set_grid_hermite(oracle_field *f, int32_t ngs, int32_t nth, int32_t nze) {
  if (!f) return -1;
  free(f->grid); f->grid = NULL; free(f->grid8); f->grid8 = NULL; f->ngs = f->nth = f->nze = 0;
  if (ngs == 0 && nth == 0 && nze == 0) return 0;
  if (ngs < 2 || nth < 2 || nze < 2) return -1;
  double *g = (double *)malloc(sizeof(double) * 8 * (size_t)ngs * nth * nze);
  if (!g) return -1;
#pragma omp parallel for collapse(2) schedule(static)
  for (int i = 0; i < ngs; ++i)
    for (int j = 0; j < nth; ++j)
      for (int k = 0; k < nze; ++k) {
        double s = (double)i / (double)(ngs - 1);
        double th = ORACLE_TWO_PI * (double)j / (double)nth;
        double ze = ORACLE_TWO_PI * (double)k / ((double)nze * (double)f->nfp);
        eval_series_mixed(f, s, th, ze, g + 8 * (((size_t)i * nth + j) * nze + k));
      }
  f->grid8 = g; f->ngs = ngs; f->nth = nth; f->nze = nze;
  return 0;
}

const double *oracle_field_grid8(const oracle_field *f) { return f->grid8; }

/* 1-D cubic Hermite basis and its x-derivative: h[corner][order] */
static void hermite_basis(double x, double h[2][2], double dh[2][2]) {
  h[0][0] = 1.0 - 3.0 * x * x + 2.0 * x * x * x;  dh[0][0] = -6.0 * x + 6.0 * x * x;
  h[1][0] = 3.0 * x * x - 2.0 * x * x * x;        dh[1][0] = 6.0 * x - 6.0 * x * x;
  h[0][1] = x - 2.0 * x * x + x * x * x;          dh[0][1] = 1.0 - 4.0 * x + 3.0 * x * x;
  h[1][1] = -x * x + x * x * x;                   dh[1][1] = -2.0 * x + 3.0 * x * x;
}

void oracle_eval_B_hermite(const oracle_field *f, double s, double th, double ze, double out[4]) {
  const double ds = 1.0 / (double)(f->ngs - 1);
  const double dth = ORACLE_TWO_PI / (double)f->nth;
  const double dze = ORACLE_TWO_PI / ((double)f->nze * (double)f->nfp);
  double us = s * (double)(f->ngs - 1), cs = floor(us);
  if (!(cs >= 0.0)) cs = 0.0;                                     /* also NaN */
  if (cs > (double)(f->ngs - 2)) cs = (double)(f->ngs - 2);
  const int64_t ci = (int64_t)cs;
  const double x = us - cs;
  double ut = th * ((double)f->nth / ORACLE_TWO_PI), ct = floor(ut), y = ut - ct;
  double uz = ze * ((double)f->nze * (double)f->nfp / ORACLE_TWO_PI), cz = floor(uz), z = uz - cz;
  double rj = fmod(ct, (double)f->nth); if (rj < 0.0) rj += (double)f->nth;
  double rk = fmod(cz, (double)f->nze); if (rk < 0.0) rk += (double)f->nze;
  const int64_t cj = (int64_t)rj, ck = (int64_t)rk;
  double hs[2][2], dhs[2][2], ht[2][2], dht[2][2], hz[2][2], dhz[2][2];
  hermite_basis(x, hs, dhs); hermite_basis(y, ht, dht); hermite_basis(z, hz, dhz);
  const double sc[2][3] = {{1.0, 1.0, 1.0}, {ds, dth, dze}};     /* slope scaling by the cell widths */
  double B = 0.0, Bs = 0.0, Bt = 0.0, Bz = 0.0;
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b)
      for (int c = 0; c < 2; ++c) {
        const int64_t i = ci + a, j = (cj + b) % f->nth, k = (ck + c) % f->nze;
        const double *D = f->grid8 + 8 * (((size_t)i * f->nth + j) * f->nze + k);
        /* D index by derivative orders (p, q, r): f 0, f_s 1, f_th 2, f_ze 3, f_s_th 4, f_s_ze 5, f_th_ze 6, all 7 */
        static const int idx[2][2][2] = {{{0, 3}, {2, 6}}, {{1, 5}, {4, 7}}};
        for (int p = 0; p < 2; ++p)
          for (int q = 0; q < 2; ++q)
            for (int r = 0; r < 2; ++r) {
              const double v = D[idx[p][q][r]] * sc[p][0] * sc[q][1] * sc[r][2];
              B += v * hs[a][p] * ht[b][q] * hz[c][r];
              Bs += v * dhs[a][p] * ht[b][q] * hz[c][r] / ds;
              Bt += v * hs[a][p] * dht[b][q] * hz[c][r] / dth;
              Bz += v * hs[a][p] * ht[b][q] * dhz[c][r] / dze;
            }
      }
  out[0] = B; out[1] = Bs; out[2] = Bt; out[3] = Bz;
}

void oracle_eval_B(const oracle_field *f, double s, double th, double ze, double out[4]) {
  if (f->grid8) { oracle_eval_B_hermite(f, s, th, ze, out); return; }
  if (f->grid) oracle_eval_B_grid(f, s, th, ze, out);
  else oracle_eval_B_sum(f, s, th, ze, out);
}

/* NEXT-4: the covariant radial component K(s, theta, zeta) of B = G grad zeta + I grad theta + K grad psi. */
void oracle_eval_K(const oracle_field *f, double s, double th, double ze, double out[4]) {
  if (!f->kmnc && !f->kmns) { out[0] = out[1] = out[2] = out[3] = 0.0; return; }
  eval_series(f, f->kmnc, f->kmns, s, th, ze, out);
}

void oracle_eval_profiles(const oracle_field *f, double s, double out[6]) {
  int32_t i0; double w[4], dw[4];
  oracle_lagrange(f->ns, s, &i0, w, dw);
  interp(f->G, 1, i0, w, dw, &out[0], &out[1]);
  interp(f->I, 1, i0, w, dw, &out[2], &out[3]);
  interp(f->iota, 1, i0, w, dw, &out[4], &out[5]);
}

/* ---- O3: shear-Alfven perturbation, Phi and alpha with E_par = 0 (A14) ----------------- */
void oracle_eval_pert(const oracle_field *f, double s, double th, double ze, double t, double out[9]) {
  for (int i = 0; i < 9; ++i) out[i] = 0.0;
  if (f->nk == 0) return;
  int32_t i0; double w[4], dw[4];
  oracle_lagrange(f->ns, s, &i0, w, dw);
  double G, Gs, I, Is, io, ios;
  interp(f->G, 1, i0, w, dw, &G, &Gs);
  interp(f->I, 1, i0, w, dw, &I, &Is);
  interp(f->iota, 1, i0, w, dw, &io, &ios);
  double Phi = 0, Phi_s = 0, Phi_th = 0, Phi_ze = 0, al = 0, al_s = 0, al_th = 0, al_ze = 0, al_t = 0;
  for (int k = 0; k < f->nk; ++k) {
    double ph, ph_s;
    interp(f->phihat + k, f->nk, i0, w, dw, &ph, &ph_s);
    double m = (double)f->mode_m[k], n = (double)f->mode_n[k], om = f->mode_omega[k];
    double ang = m * th - n * ze + om * t + f->mode_phase[k];
    double sn = sin(ang), c = cos(ang);
    /* alpha_hat = -Phi_hat (iota m - n) / (omega (G + iota I)) */
    double N = io * m - n, N_s = ios * m;
    double Dn = om * (G + io * I), Dn_s = om * (Gs + ios * I + io * Is);
    double ah = -ph * N / Dn;
    double ah_s = -(ph_s * N / Dn + ph * N_s / Dn - ph * N * Dn_s / (Dn * Dn));
    Phi += ph * sn;
    Phi_s += ph_s * sn;
    Phi_th += m * ph * c;
    Phi_ze += -n * ph * c;
    al += ah * sn;
    al_s += ah_s * sn;
    al_th += m * ah * c;
    al_ze += -n * ah * c;
    al_t += om * ah * c;
  }
  out[0] = Phi; out[1] = Phi_s / f->psi0; out[2] = Phi_th; out[3] = Phi_ze;
  out[4] = al; out[5] = al_s / f->psi0; out[6] = al_th; out[7] = al_ze; out[8] = al_t;
}

/* ---- O4: guiding-centre equations in Boozer coordinates (A4) ------------------------
 * Euler-Lagrange equations of L = q(psi + rho_c I) thdot + q(rho_c G - chi) zedot - H,
 * rho_c = m v/(q B) + alpha, H = m v^2/2 + mu B + q Phi, chi' = iota, covariant radial component dropped. */
void oracle_rhs(const oracle_field *f, double mass, double charge, double mu, double v_ref,
                double t, const double y[4], double dydt[4]) {
  if (f->kmnc || f->kmns) { oracle_rhs_general(f, mass, charge, mu, v_ref, t, y, dydt); return; }
  double s = y[0], th = y[1], ze = y[2], v = y[3] * v_ref;
  double fb[4], pr[6], pt[9];
  oracle_eval_B(f, s, th, ze, fb);
  oracle_eval_profiles(f, s, pr);
  oracle_eval_pert(f, s, th, ze, t, pt);
  double psi0 = f->psi0;
  double B = fb[0], B_psi = fb[1] / psi0, B_th = fb[2], B_ze = fb[3];
  double G = pr[0], Gp = pr[1] / psi0, I = pr[2], Ip = pr[3] / psi0, iota = pr[4];
  double Phi_psi = pt[1], Phi_th = pt[2], Phi_ze = pt[3];
  double al = pt[4], al_psi = pt[5], al_th = pt[6], al_ze = pt[7], al_t = pt[8];

  double rho = mass * v / (charge * B);
  double rho_c = rho + al;
  double F = mass * v * v / B + mu;
  double a = 1.0 + rho_c * Ip + al_psi * I;
  double b = iota - rho_c * Gp - al_psi * G;
  double D = a * G + b * I;
  double C = al_th * G - al_ze * I;
  double h_psi = F / charge * B_psi + Phi_psi;
  double h_th = F / charge * B_th + Phi_th;
  double h_ze = F / charge * B_ze + Phi_ze;
  double psidot = (I * h_ze - G * h_th + C * v * B) / D;
  double thdot = (b * v * B + G * h_psi) / D;
  double zedot = (a * v * B - I * h_psi) / D;
  double Lam = a * B_ze + b * B_th + C * B_psi;
  double mvdot = (-mu * B * Lam - charge * B * (a * Phi_ze + b * Phi_th + C * Phi_psi)
                  + (mass * v / B) * (B_psi * (I * Phi_ze - G * Phi_th) + Phi_psi * (G * B_th - I * B_ze))) / D
                 - charge * B * al_t;
  dydt[0] = psidot / psi0;
  dydt[1] = thdot;
  dydt[2] = zedot;
  dydt[3] = mvdot / mass / v_ref;
}

/* ---- O4, general form (NEXT-4: K kept) ---------------------------------------------------------------
 * z = (psi, theta, zeta, v).  A*_psi = rho_c K, A*_theta = psi + rho_c I, A*_zeta = rho_c G - chi, A*_v = 0
 * (all times q).  omega_ij = d_i A*_j - d_j A*_i.  Equations: q sum_j omega_ij zdot_j = d_i H + q d_t A*_i with
 * H = m v^2/2 + mu B + q Phi.  K_psi never appears (d_psi A*_psi cancels). */
void oracle_rhs_general(const oracle_field *f, double mass, double charge, double mu, double v_ref,
                        double t, const double y[4], double dydt[4]) {
  double s = y[0], th = y[1], ze = y[2], v = y[3] * v_ref;
  double fb[4], fk[4], pr[6], pt[9];
  oracle_eval_B(f, s, th, ze, fb);
  oracle_eval_K(f, s, th, ze, fk);
  oracle_eval_profiles(f, s, pr);
  oracle_eval_pert(f, s, th, ze, t, pt);
  double psi0 = f->psi0, q = charge;
  double B = fb[0];
  double dB[3] = {fb[1] / psi0, fb[2], fb[3]};                 /* d/dpsi, d/dtheta, d/dzeta */
  double K = fk[0], dK[3] = {fk[1] / psi0, fk[2], fk[3]};
  double G = pr[0], Gp = pr[1] / psi0, I = pr[2], Ip = pr[3] / psi0, iota = pr[4];
  double dPhi[3] = {pt[1], pt[2], pt[3]};
  double al = pt[4], dal[3] = {pt[5], pt[6], pt[7]}, al_t = pt[8];
  double rho = mass * v / (q * B), rho_c = rho + al;
  double r[3], rv = mass / (q * B);                            /* d rho_c / d(psi, theta, zeta), d rho_c / dv */
  for (int x = 0; x < 3; ++x) r[x] = -rho * dB[x] / B + dal[x];
  /* dA[i][j] = d A*_j / d z_i  (i, j over psi, theta, zeta, v) */
  double dA[4][4];
  for (int i = 0; i < 3; ++i) {
    dA[i][0] = r[i] * K + rho_c * dK[i];
    dA[i][1] = r[i] * I + (i == 0 ? 1.0 + rho_c * Ip : 0.0);
    dA[i][2] = r[i] * G + (i == 0 ? rho_c * Gp - iota : 0.0);
    dA[i][3] = 0.0;
  }
  dA[3][0] = rv * K; dA[3][1] = rv * I; dA[3][2] = rv * G; dA[3][3] = 0.0;
  double Mx[4][5];
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j) Mx[i][j] = q * (dA[i][j] - dA[j][i]);
  double At[3] = {al_t * K, al_t * I, al_t * G};               /* d A*_i / dt */
  for (int i = 0; i < 3; ++i) Mx[i][4] = mu * dB[i] + q * dPhi[i] + q * At[i];
  Mx[3][4] = mass * v;
  /* Gaussian elimination with partial pivoting on rows scaled to unit maximum */
  for (int i = 0; i < 4; ++i) {
    double big = 0.0;
    for (int j = 0; j < 4; ++j) big = fmax(big, fabs(Mx[i][j]));
    for (int j = 0; j < 5; ++j) Mx[i][j] /= big;
  }
  for (int c = 0; c < 4; ++c) {
    int piv = c;
    for (int i = c + 1; i < 4; ++i) if (fabs(Mx[i][c]) > fabs(Mx[piv][c])) piv = i;
    for (int j = 0; j < 5; ++j) { double tmp = Mx[c][j]; Mx[c][j] = Mx[piv][j]; Mx[piv][j] = tmp; }
    for (int i = c + 1; i < 4; ++i) {
      double fct = Mx[i][c] / Mx[c][c];
      for (int j = c; j < 5; ++j) Mx[i][j] -= fct * Mx[c][j];
    }
  }
  double zd[4];
  for (int i = 3; i >= 0; --i) {
    double acc = Mx[i][4];
    for (int j = i + 1; j < 4; ++j) acc -= Mx[i][j] * zd[j];
    zd[i] = acc / Mx[i][i];
  }
  dydt[0] = zd[0] / psi0;
  dydt[1] = zd[1];
  dydt[2] = zd[2];
  dydt[3] = zd[3] / v_ref;
}

/* ---- O5: Dormand-Prince 5(4), FSAL ---------------------------------------------------- */
static const double DP_C[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
static const double DP_A[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1.0 / 5.0, 0, 0, 0, 0, 0},
    {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0}};
static const double DP_E[7] = {71.0 / 57600.0, 0.0, -71.0 / 16695.0, 71.0 / 1920.0,
                               -17253.0 / 339200.0, 22.0 / 525.0, -1.0 / 40.0};
static const double DP_D[7] = {-12715105075.0 / 11282082432.0, 0.0, 87487479700.0 / 32700410799.0,
                               -10690763975.0 / 1880347072.0, 701980252875.0 / 199316789632.0,
                               -1453857185.0 / 822651844.0, 69997945.0 / 29380423.0};

void oracle_dp5_attempt_fn(oracle_rhs_fn fn, void *ctx, double t, const double y[4], const double k1[4],
                           double h, double y_new[4], double k[7][4], double delta[4]) {
  for (int c = 0; c < 4; ++c) k[0][c] = k1[c];
  double ys[4];
  for (int i = 1; i < 7; ++i) {                      /* stages 2..7; stage 7 is evaluated at y_new */
    for (int c = 0; c < 4; ++c) {
      double acc = 0.0;
      for (int j = 0; j < i; ++j) acc += DP_A[i][j] * k[j][c];
      ys[c] = y[c] + h * acc;
    }
    fn(ctx, t + DP_C[i] * h, ys, k[i]);
  }
  for (int c = 0; c < 4; ++c) {
    y_new[c] = ys[c];                                /* row 7 of A is the 5th-order weights */
    double e = 0.0;
    for (int j = 0; j < 7; ++j) e += DP_E[j] * k[j][c];
    delta[c] = h * e;
  }
}

typedef struct { const oracle_field *f; double mass, charge, mu, v_ref; } gc_ctx;

static void gc_rhs_fn(void *ctx, double t, const double y[4], double dydt[4]) {
  const gc_ctx *g = (const gc_ctx *)ctx;
  oracle_rhs(g->f, g->mass, g->charge, g->mu, g->v_ref, t, y, dydt);
}

void oracle_dp5_attempt(const oracle_field *f, double mass, double charge, double mu, double v_ref,
                        double t, const double y[4], const double k1[4], double h,
                        double y_new[4], double k[7][4], double delta[4]) {
  gc_ctx g = {f, mass, charge, mu, v_ref};
  oracle_dp5_attempt_fn(gc_rhs_fn, &g, t, y, k1, h, y_new, k, delta);
}

/* ---- O8: continuous extension of the step --------------------------------------------------------- */
static void dense_and_slope(const double y[4], const double y_new[4], const double k[7][4], double h,
                            double tau, double y_tau[4], double dy_dtau[4]) {
  double sg = 1.0 - tau;
  for (int c = 0; c < 4; ++c) {
    double r1 = y[c], r2 = y_new[c] - y[c];
    double r3 = h * k[0][c] - r2;
    double r4 = r2 - h * k[6][c] - r3;
    double r5 = 0.0;
    for (int j = 0; j < 7; ++j) r5 += DP_D[j] * k[j][c];
    r5 *= h;
    double P4 = r4 + sg * r5, dP4 = -r5;
    double P3 = r3 + tau * P4, dP3 = P4 + tau * dP4;
    double P2 = r2 + sg * P3, dP2 = -P3 + sg * dP3;
    y_tau[c] = r1 + tau * P2;
    dy_dtau[c] = P2 + tau * dP2;
  }
}

void oracle_dp5_dense(const double y[4], const double y_new[4], const double k[7][4], double h,
                      double tau, double y_tau[4]) {
  double d[4];
  dense_and_slope(y, y_new, k, h, tau, y_tau, d);
}

/* ---- O6: error norm and step-size factors (Press 2007 style; A10) ---------------------------------- */
double oracle_err_norm(const double y[4], const double y_new[4], const double delta[4],
                       double rtol, double atol) {
  double acc = 0.0;
  for (int c = 0; c < 4; ++c) {
    double sk = atol + rtol * fmax(fabs(y[c]), fabs(y_new[c]));
    double r = delta[c] / sk;
    acc += r * r;
  }
  return sqrt(acc / 4.0);
}

#define CTRL_SAFETY 0.9
#define CTRL_MINSCALE 0.2
#define CTRL_MAXSCALE 10.0
#define CTRL_ALPHA 0.2          /* beta = 0: alpha = 0.2 - 0.75 beta */

double oracle_scale_accept(double err) {
  if (err == 0.0) return CTRL_MAXSCALE;
  double sc = CTRL_SAFETY * pow(err, -CTRL_ALPHA);
  if (sc < CTRL_MINSCALE) sc = CTRL_MINSCALE;
  if (sc > CTRL_MAXSCALE) sc = CTRL_MAXSCALE;
  return sc;
}

double oracle_scale_reject(double err) {
  if (!isfinite(err)) return CTRL_MINSCALE;
  double sc = CTRL_SAFETY * pow(err, -CTRL_ALPHA);
  return sc > CTRL_MINSCALE ? sc : CTRL_MINSCALE;
}

static int all_finite4(const double v[4]) {
  return isfinite(v[0]) && isfinite(v[1]) && isfinite(v[2]) && isfinite(v[3]);
}

/* O8: one crossing of component `comp` through `target` inside the accepted step (t, y) -> (t+h, y_new): root of
 * the continuous extension by 8 bisections and Newton, then the record (id, t + tau h, s, theta mod 2 pi). */
static void record_crossing(int64_t id, double t, double h, const double y[4], const double y_new[4],
                            const double k[7][4], int comp, double target, double tol,
                            double *buf, int64_t cap, int64_t *count) {
  const double TWO_PI = 6.283185307179586476925286766559;
  double lo = 0.0, hi = 1.0, yt[4], dy[4];
  double glo = y[comp] - target;
  for (int it = 0; it < 8; ++it) {                                  /* bisection to bracket */
    double mid = 0.5 * (lo + hi);
    dense_and_slope(y, y_new, k, h, mid, yt, dy);
    double g = yt[comp] - target;
    if ((g < 0.0) == (glo < 0.0) && g != 0.0) { lo = mid; glo = g; } else { hi = mid; }
  }
  double tau = 0.5 * (lo + hi);
  for (int it = 0; it < 20; ++it) {                                 /* Newton polish */
    dense_and_slope(y, y_new, k, h, tau, yt, dy);
    double g = yt[comp] - target;
    if (fabs(g) < tol || dy[comp] == 0.0) break;
    double tn = tau - g / dy[comp];
    if (tn < lo) tn = lo;
    if (tn > hi) tn = hi;
    tau = tn;
  }
  dense_and_slope(y, y_new, k, h, tau, yt, dy);
  int64_t slot;
#pragma omp atomic capture
  slot = (*count)++;
  if (slot < cap) {
    double thm = fmod(yt[1], TWO_PI);
    if (thm < 0.0) thm += TWO_PI;
    buf[slot * 4 + 0] = (double)id;
    buf[slot * 4 + 1] = t + tau * h;
    buf[slot * 4 + 2] = yt[0];
    buf[slot * 4 + 3] = thm;
  }
}

/* O8: record every crossing of zeta = 2 pi k inside the accepted step (t, y) -> (t+h, y_new). */
static void poincare_step(int64_t id, double t, double h, const double y[4], const double y_new[4],
                          const double k[7][4], double *buf, int64_t cap, int64_t *count) {
  const double TWO_PI = 6.283185307179586476925286766559;
  double k0 = floor(y[2] / TWO_PI), k1 = floor(y_new[2] / TWO_PI);
  if (k0 == k1) return;
  double kfirst, klast, kstep;
  if (k1 > k0) { kfirst = k0 + 1.0; klast = k1; kstep = 1.0; }        /* planes crossed going up   */
  else { kfirst = k0; klast = k1 + 1.0; kstep = -1.0; }               /* planes crossed going down */
  for (double kp = kfirst; kstep > 0 ? kp <= klast : kp >= klast; kp += kstep) {
    double target = TWO_PI * kp;
    record_crossing(id, t, h, y, y_new, k, 2, target, 1e-12 * fmax(1.0, fabs(target)), buf, cap, count);
  }
}

/* O8b (NEXT-1; "trapped particle Poincare map"): the bounce section v_par = 0.  A step whose end
 * values of u = v_par / v_ref have opposite signs (or that ends exactly on 0 from a nonzero start) holds one
 * crossing; both directions count; u is O(1), so the root tolerance is 1e-12 absolute. */
static void bounce_step(int64_t id, double t, double h, const double y[4], const double y_new[4],
                        const double k[7][4], double *buf, int64_t cap, int64_t *count) {
  if (!((y[3] < 0.0 && y_new[3] >= 0.0) || (y[3] > 0.0 && y_new[3] <= 0.0))) return;
  record_crossing(id, t, h, y, y_new, k, 3, 0.0, 1e-12, buf, cap, count);
}

/* ---- O5-O8: the trace -------------------------------------------------------------------------------- */
/* O9 (NEXT-1): time of sample j.  One fused multiply-add, so that both implementations round it alike. */
static double sample_time(double sample_t0, double sample_dt, int64_t j) { return fma((double)j, sample_dt, sample_t0); }

static int trace_impl(const oracle_field *f, const oracle_trace_params *p, int64_t n,
                      const double *s0, const double *th0, const double *ze0, const double *vpar0,
                      const double *mu, double *h_inout,
                      double *y_out, double *t_out, int32_t *status,
                      int32_t *n_acc_out, int32_t *n_rej_out, int32_t *n_forced_out,
                      double *poincare, int64_t *poincare_count,
                      double *traj, int64_t *traj_count,
                      double sample_t0, double sample_dt, int64_t nsamp, double *samples, int32_t *nsampled) {
  if (!f || !p || n < 0 || !(p->v_ref > 0.0) || !(p->h0 > 0.0) || p->h_min < 0.0) return -1;
  if (nsamp > 0 && (!samples || !(sample_dt > 0.0))) return -1;
  if (poincare_count) *poincare_count = 0;
  int64_t pcap = (poincare && poincare_count) ? p->poincare_capacity : 0;
  int64_t tcap = (traj && traj_count) ? p->traj_capacity : 0;

#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t i = 0; i < n; ++i) {
    double y[4] = {s0[i], th0[i], ze0[i], vpar0[i] / p->v_ref};
    double t = p->t0, h = (h_inout && h_inout[i] > 0.0) ? h_inout[i] : p->h0;
    if (h < p->h_min) h = p->h_min;
    double k[7][4], k1[4], y_new[4], delta[4];
    int64_t attempts = 0;
    int32_t n_acc = 0, n_rej = 0, n_forced = 0, st = -1;
    int prev_rejected = 0;
    int64_t ntraj = 0;
    /* O9: next sample index = first j with tau_j >= t0; a sample that falls on t0 is the initial state */
    int64_t jn = 0;
    if (nsamp > 0) {
      while (jn < nsamp && sample_time(sample_t0, sample_dt, jn) < t) ++jn;
      if (jn < nsamp && sample_time(sample_t0, sample_dt, jn) == t) {
        for (int c = 0; c < 4; ++c) samples[((size_t)c * nsamp + jn) * n + i] = c == 3 ? y[3] * p->v_ref : y[c];
        ++jn;
      }
    }
    oracle_rhs(f, p->mass, p->charge, mu[i], p->v_ref, t, y, k1);
    if (!all_finite4(y) || !all_finite4(k1)) st = 4;
    else if (!(t < p->t_max)) st = 0;
    while (st < 0) {
      double h_try = h;
      int clipped = 0;
      if (t + h_try >= p->t_max) { h_try = p->t_max - t; clipped = 1; }       /* end clip */
      if (!(t + h_try > t)) { st = 4; break; }                                /* step underflow */
      int forced = prev_rejected && p->h_min > 0.0 && h == p->h_min;
      oracle_dp5_attempt(f, p->mass, p->charge, mu[i], p->v_ref, t, y, k1, h_try, y_new, k, delta);
      ++attempts;
      double err = oracle_err_norm(y, y_new, delta, p->rtol, p->atol);
      int finite = all_finite4(y_new) && all_finite4(k[6]) && isfinite(err);
      int accept;
      if (forced) {
        if (!finite) { st = 4; break; }
        accept = 1;
      } else {
        accept = finite && err <= 1.0;
      }
      if (accept) {
        double sc = oracle_scale_accept(err);
        double h_next = prev_rejected ? h_try * fmin(sc, 1.0) : h_try * sc;
        if (pcap > 0) {
          if (p->section == 1) bounce_step(i, t, h_try, y, y_new, (const double(*)[4])k, poincare, pcap, poincare_count);
          else poincare_step(i, t, h_try, y, y_new, (const double(*)[4])k, poincare, pcap, poincare_count);
        }
        const double t_new = clipped ? p->t_max : t + h_try;
        while (jn < nsamp) {                   /* O9: samples with t < tau_j <= t_new from the continuous extension */
          double tj = sample_time(sample_t0, sample_dt, jn), ys[4];
          if (tj > t_new) break;
          oracle_dp5_dense(y, y_new, (const double(*)[4])k, h_try, (tj - t) / h_try, ys);
          for (int c = 0; c < 4; ++c) samples[((size_t)c * nsamp + jn) * n + i] = c == 3 ? ys[3] * p->v_ref : ys[c];
          ++jn;
        }
        /* O7b: refined loss point, taken after the samples and records of the step (they run to its end) */
        const int lost_now = y_new[0] >= p->s_loss;
        double t_rep = t_new, y_rep[4] = {y_new[0], y_new[1], y_new[2], y_new[3]};
        if (lost_now && p->refine_loss && y[0] < p->s_loss) {
          double lo = 0.0, hi = 1.0, yt[4], dyt[4];
          for (int it = 0; it < 8; ++it) {
            double mid = 0.5 * (lo + hi);
            dense_and_slope(y, y_new, (const double(*)[4])k, h_try, mid, yt, dyt);
            if (yt[0] < p->s_loss) lo = mid; else hi = mid;
          }
          double tau = 0.5 * (lo + hi);
          for (int it = 0; it < 20; ++it) {
            dense_and_slope(y, y_new, (const double(*)[4])k, h_try, tau, yt, dyt);
            double g = yt[0] - p->s_loss;
            if (fabs(g) < 1e-14 || dyt[0] == 0.0) break;
            double tn = tau - g / dyt[0];
            tau = tn < lo ? lo : (tn > hi ? hi : tn);
          }
          dense_and_slope(y, y_new, (const double(*)[4])k, h_try, tau, y_rep, dyt);
          t_rep = t + tau * h_try;
        }
        t = t_new;
        for (int c = 0; c < 4; ++c) { y[c] = y_new[c]; k1[c] = k[6][c]; }
        ++n_acc;
        if (forced) ++n_forced;
        prev_rejected = 0;
        if (!clipped) h = h_next;              /* a clipped last step keeps the unclipped proposal */
        if (h < p->h_min) h = p->h_min;
        if (ntraj < tcap) {
          double *r = traj + ((size_t)i * tcap + ntraj) * 5;
          r[0] = t; r[1] = y[0]; r[2] = y[1]; r[3] = y[2]; r[4] = y[3];
        }
        ++ntraj;
        /* O7 stop rules, in this order */
        if (lost_now) { st = 1; t = t_rep; for (int c = 0; c < 4; ++c) y[c] = y_rep[c]; }
        else if (y[0] <= p->s_min) st = 2;
        else if (clipped) st = 0;
        else if (attempts >= p->max_steps) st = 3;
      } else {
        ++n_rej;
        h = h_try * oracle_scale_reject(err);
        if (h < p->h_min) h = p->h_min;
        prev_rejected = 1;
        if (attempts >= p->max_steps) st = 3;
      }
    }
    y_out[0 * n + i] = y[0];
    y_out[1 * n + i] = y[1];
    y_out[2 * n + i] = y[2];
    y_out[3 * n + i] = y[3] * p->v_ref;        /* v_par back in m/s */
    t_out[i] = t;
    status[i] = st;
    if (h_inout) h_inout[i] = h;
    if (n_acc_out) n_acc_out[i] = n_acc;
    if (n_rej_out) n_rej_out[i] = n_rej;
    if (n_forced_out) n_forced_out[i] = n_forced;
    if (traj_count) traj_count[i] = ntraj;
    if (nsampled) nsampled[i] = (int32_t)jn;
  }
  return 0;
}

int oracle_trace(const oracle_field *f, const oracle_trace_params *p, int64_t n,
                 const double *s0, const double *th0, const double *ze0, const double *vpar0,
                 const double *mu, double *h_inout,
                 double *y_out, double *t_out, int32_t *status,
                 int32_t *n_acc_out, int32_t *n_rej_out, int32_t *n_forced_out,
                 double *poincare, int64_t *poincare_count,
                 double *traj, int64_t *traj_count) {
  return trace_impl(f, p, n, s0, th0, ze0, vpar0, mu, h_inout, y_out, t_out, status, n_acc_out, n_rej_out,
                    n_forced_out, poincare, poincare_count, traj, traj_count, 0.0, 0.0, 0, NULL, NULL);
}

int oracle_trace_sampled(const oracle_field *f, const oracle_trace_params *p, int64_t n,
                         const double *s0, const double *th0, const double *ze0, const double *vpar0,
                         const double *mu, double *h_inout,
                         double *y_out, double *t_out, int32_t *status,
                         int32_t *n_acc_out, int32_t *n_rej_out, int32_t *n_forced_out,
                         double sample_t0, double sample_dt, int64_t nsamp, double *samples, int32_t *nsampled) {
  return trace_impl(f, p, n, s0, th0, ze0, vpar0, mu, h_inout, y_out, t_out, status, n_acc_out, n_rej_out,
                    n_forced_out, NULL, NULL, NULL, NULL, sample_t0, sample_dt, nsamp, samples, nsampled);
}

/* A17: canonical toroidal momentum P_zeta = q ((rho + alpha) G - chi(s)), rho = m v_par / (q B), chi' = iota with
 * respect to psi; chi is given at the radial nodes and interpolated like every other profile (O1). */
double oracle_pzeta(const oracle_field *f, double mass, double charge, const double *chi_nodes,
                    double s, double th, double ze, double vpar, double t) {
  double fb[4], pr[6], pt[9] = {0};
  int32_t i0;
  double w[4], dw[4];
  oracle_eval_B(f, s, th, ze, fb);
  oracle_eval_profiles(f, s, pr);
  oracle_eval_pert(f, s, th, ze, t, pt);
  oracle_lagrange(f->ns, s, &i0, w, dw);
  double chi = 0.0;
  for (int a = 0; a < 4; ++a) chi += w[a] * chi_nodes[i0 + a];
  double rho = mass * vpar / (charge * fb[0]);
  return charge * ((rho + pt[4]) * pr[0] - chi);
}

/* ---- NEXT-3 ("A symplectic integrator for non-canonical guiding-center orbits uses the
 * explicit-implicit Euler scheme of (Albert et al., 2020)"; Fig. 1 left; reading A28 of DESIGN.md).
 *
 * Albert et al. 2020 is not in the container; the scheme is restated from what the sentence fixes.  For a static field
 * with K = 0 and no perturbation the guiding-centre Lagrangian of O4,
 *     L = q (psi + rho I) thetadot + q (rho G - chi) zetadot - H,     rho = m v_par / (q B),  H = m v_par^2 / 2 + mu B,
 * is already of the form p_theta thetadot + p_zeta zetadot - H with the canonical momenta
 *     p_theta = q (psi0 s + rho I(s)),     p_zeta = q (rho G(s) - chi(s)),
 * so (theta, zeta, p_theta, p_zeta) are canonical coordinates and s is a parameter fixed by them ("non-canonical":
 * the state carried is z = (s, theta, zeta, p_zeta)).  With rho(s, p_zeta) = (p_zeta / q + chi(s)) / G(s),
 *     H(s, theta, zeta, p_zeta) = (q rho B)^2 / (2 m) + mu B,          p_theta(s, p_zeta) = q (psi0 s + rho I),
 * the symplectic ("explicit-implicit") Euler step of size h, implicit in the momenta and explicit in the angles, is
 *     p_theta(s', p_zeta') - p_theta(s, p_zeta) + h dH/dtheta = 0        (1)   derivatives of H at constant s, p_zeta
 *     p_zeta' - p_zeta                          + h dH/dzeta  = 0        (2)   taken at (s', theta, zeta, p_zeta')
 *     theta' = theta + h (dH/ds) / (dp_theta/ds)                          (3)
 *     zeta'  = zeta  + h [ dH/dp_zeta - (dH/ds) (dp_theta/dp_zeta) / (dp_theta/ds) ]          (4)
 * (the chain rule through s(theta, zeta, p_theta, p_zeta) turns the canonical dK/dp_theta, dK/dp_zeta, dK/dtheta,
 * dK/dzeta of K = H(s(..), ..) into these; p_theta does not depend on the angles here).  (1), (2) are solved for
 * (s', p_zeta') by Newton's method on the scaled unknowns x = (s, p_zeta / (q psi0)) with a central-difference
 * Jacobian (step 1e-6), started from the old values, until max |dx_i| <= newton_tol max(1, |x_i|); at most 50
 * iterations, failure or a non-finite value ends the particle with status 4.  chi(s) is supplied at the radial
 * nodes (as for oracle_pzeta) and interpolated by O1, and d chi / d s of THAT interpolant is what the scheme uses
 * where the equations of motion have psi0 iota: the map is then exactly symplectic within a radial cell.
 * Stop rules after every step as O7: s >= s_loss -> 1, s <= s_min -> 2; nsteps steps done -> 0. */
typedef struct {
  const oracle_field *f;
  const double *chi_nodes;
  double mass, charge, mu;
} sym_ctx;

/* H and p_theta with their first partial derivatives at (s, theta, zeta, p_zeta). */
static void sym_eval(const sym_ctx *c, double s, double th, double ze, double pz,
                     double *H, double dH[4] /* d/ds, d/dtheta, d/dzeta, d/dp_zeta */,
                     double *ptheta, double *dpth_ds, double *dpth_dpz, double *vpar) {
  const oracle_field *f = c->f;
  const double q = c->charge, m = c->mass;
  double fb[4], pr[6];
  oracle_eval_B(f, s, th, ze, fb);
  oracle_eval_profiles(f, s, pr);
  int32_t i0; double w[4], dw[4], chi, chi_s;
  oracle_lagrange(f->ns, s, &i0, w, dw);
  interp(c->chi_nodes, 1, i0, w, dw, &chi, &chi_s);
  const double B = fb[0], Bs = fb[1], Bth = fb[2], Bze = fb[3];
  const double G = pr[0], Gs = pr[1], I = pr[2], Is = pr[3];
  const double rho = (pz / q + chi) / G;
  const double rho_s = (chi_s - rho * Gs) / G;
  const double rho_pz = 1.0 / (q * G);
  const double e = q * q * rho * rho * B / m + c->mu;        /* dH/dB */
  *H = q * q * rho * rho * B * B / (2.0 * m) + c->mu * B;
  dH[0] = q * q * rho * rho_s * B * B / m + e * Bs;
  dH[1] = e * Bth;
  dH[2] = e * Bze;
  dH[3] = q * q * rho * rho_pz * B * B / m;
  *ptheta = q * (f->psi0 * s + rho * I);
  *dpth_ds = q * (f->psi0 + rho_s * I + rho * Is);
  *dpth_dpz = q * rho_pz * I;
  *vpar = q * rho * B / m;
}

/* residuals of (1), (2) in units of q psi0 at the scaled unknowns x = (s, p_zeta / (q psi0)) */
static void sym_residual(const sym_ctx *c, double th, double ze, double pth_old, double pz_old, double h,
                         const double x[2], double F[2]) {
  const double unit = c->charge * c->f->psi0;
  double H, dH[4], pth, d1, d2, v;
  sym_eval(c, x[0], th, ze, x[1] * unit, &H, dH, &pth, &d1, &d2, &v);
  F[0] = (pth - pth_old + h * dH[1]) / unit;
  F[1] = (x[1] * unit - pz_old + h * dH[2]) / unit;
}

int oracle_symplectic_step(const oracle_field *f, double mass, double charge, double mu, const double *chi_nodes,
                           double h, double newton_tol, double z[4] /* s, theta, zeta, p_zeta: in and out */,
                           int32_t *iterations) {
  sym_ctx c = {f, chi_nodes, mass, charge, mu};
  const double unit = charge * f->psi0;
  double H, dH[4], pth_old, d1, d2, v;
  sym_eval(&c, z[0], z[1], z[2], z[3], &H, dH, &pth_old, &d1, &d2, &v);
  double x[2] = {z[0], z[3] / unit};
  int ok = 0, it = 0;
  for (it = 1; it <= 50; ++it) {
    double F[2], J[2][2];
    sym_residual(&c, z[1], z[2], pth_old, z[3], h, x, F);
    for (int j = 0; j < 2; ++j) {
      const double e = 1e-6;
      double xp[2] = {x[0], x[1]}, xm[2] = {x[0], x[1]}, Fp[2], Fm[2];
      xp[j] += e; xm[j] -= e;
      sym_residual(&c, z[1], z[2], pth_old, z[3], h, xp, Fp);
      sym_residual(&c, z[1], z[2], pth_old, z[3], h, xm, Fm);
      J[0][j] = (Fp[0] - Fm[0]) / (2.0 * e);
      J[1][j] = (Fp[1] - Fm[1]) / (2.0 * e);
    }
    const double det = J[0][0] * J[1][1] - J[0][1] * J[1][0];
    const double dx0 = -(J[1][1] * F[0] - J[0][1] * F[1]) / det;
    const double dx1 = -(-J[1][0] * F[0] + J[0][0] * F[1]) / det;
    if (!isfinite(dx0) || !isfinite(dx1)) break;
    x[0] += dx0; x[1] += dx1;
    if (fabs(dx0) <= newton_tol * fmax(1.0, fabs(x[0])) && fabs(dx1) <= newton_tol * fmax(1.0, fabs(x[1]))) {
      ok = 1;
      break;
    }
  }
  if (iterations) *iterations = it;
  if (!ok) return -1;
  sym_eval(&c, x[0], z[1], z[2], x[1] * unit, &H, dH, &pth_old, &d1, &d2, &v);   /* partials at (s', theta, zeta, p_zeta') */
  z[1] = z[1] + h * dH[0] / d1;
  z[2] = z[2] + h * (dH[3] - dH[0] * d2 / d1);
  z[0] = x[0];
  z[3] = x[1] * unit;
  return 0;
}

/* p_zeta of a state given as (s, theta, zeta, v_par) and back (static field: no alpha). */
double oracle_symplectic_pzeta(const oracle_field *f, double mass, double charge, const double *chi_nodes,
                               double s, double th, double ze, double vpar) {
  return oracle_pzeta(f, mass, charge, chi_nodes, s, th, ze, vpar, 0.0);
}

double oracle_symplectic_vpar(const oracle_field *f, double mass, double charge, const double *chi_nodes,
                              double s, double th, double ze, double pz) {
  sym_ctx c = {f, chi_nodes, mass, charge, 0.0};
  double H, dH[4], pth, d1, d2, v;
  sym_eval(&c, s, th, ze, pz, &H, dH, &pth, &d1, &d2, &v);
  return v;
}

int oracle_trace_symplectic(const oracle_field *f, const oracle_symplectic_params *p, int64_t n,
                            const double *s0, const double *th0, const double *ze0, const double *vpar0,
                            const double *mu, const double *chi_nodes,
                            double *y_out, double *t_out, int32_t *status, int32_t *n_steps, int32_t *n_iter,
                            int64_t sample_stride, int64_t nsamp, double *samples, int32_t *sample_end) {
  if (!f || !p || n < 0 || !chi_nodes || f->nk > 0 || f->kmnc || f->kmns || !(p->dt > 0.0) || p->nsteps < 0 ||
      !(p->newton_tol > 0.0) || (nsamp > 0 && (sample_stride < 1 || !samples || !sample_end)))
    return -1;
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t i = 0; i < n; ++i) {
    double z[4] = {s0[i], th0[i], ze0[i], 0.0};
    z[3] = oracle_symplectic_pzeta(f, p->mass, p->charge, chi_nodes, z[0], z[1], z[2], vpar0[i]);
    double vpar = vpar0[i];
    int32_t st = 0, steps = 0, iters = 0;
    int64_t js = 0;
    if (!isfinite(z[0]) || !isfinite(z[1]) || !isfinite(z[2]) || !isfinite(z[3])) st = 4;
    if (nsamp > 0 && st == 0) {                                /* sample 0 is the initial state */
      samples[(0 * nsamp + 0) * n + i] = z[0]; samples[(1 * nsamp + 0) * n + i] = z[1];
      samples[(2 * nsamp + 0) * n + i] = z[2]; samples[(3 * nsamp + 0) * n + i] = vpar;
      js = 1;
    }
    for (int64_t k = 0; k < p->nsteps && st == 0; ++k) {
      int32_t it = 0;
      int rc = oracle_symplectic_step(f, p->mass, p->charge, mu[i], chi_nodes, p->dt, p->newton_tol, z, &it);
      iters += it;
      if (rc != 0 || !isfinite(z[0]) || !isfinite(z[1]) || !isfinite(z[2]) || !isfinite(z[3])) { st = 4; break; }
      ++steps;
      if (nsamp > 0 && js < nsamp && (k + 1) % sample_stride == 0) {     /* state after every sample_stride-th step */
        samples[(0 * nsamp + js) * n + i] = z[0]; samples[(1 * nsamp + js) * n + i] = z[1];
        samples[(2 * nsamp + js) * n + i] = z[2];
        samples[(3 * nsamp + js) * n + i] =
            oracle_symplectic_vpar(f, p->mass, p->charge, chi_nodes, z[0], z[1], z[2], z[3]);
        ++js;
      }
      if (z[0] >= p->s_loss) st = 1;
      else if (z[0] <= p->s_min) st = 2;
    }
    if (steps > 0) vpar = oracle_symplectic_vpar(f, p->mass, p->charge, chi_nodes, z[0], z[1], z[2], z[3]);
    y_out[0 * n + i] = z[0]; y_out[1 * n + i] = z[1]; y_out[2 * n + i] = z[2]; y_out[3 * n + i] = vpar;
    t_out[i] = p->t0 + (double)steps * p->dt;
    status[i] = st;
    if (n_steps) n_steps[i] = steps;
    if (n_iter) n_iter[i] = iters;
    if (nsamp > 0) sample_end[i] = (int32_t)js;
  }
  return 0;
}

/* ---- check (d): classical RK4 at fixed step -------------------------------------------------------- */
void oracle_rk4(const oracle_field *f, double mass, double charge, double v_ref, int64_t n,
                const double *s0, const double *th0, const double *ze0, const double *vpar0,
                const double *mu, double t0, double h, int64_t nsteps, double *y_out) {
#pragma omp parallel for schedule(dynamic, 1)
  for (int64_t i = 0; i < n; ++i) {
    double y[4] = {s0[i], th0[i], ze0[i], vpar0[i] / v_ref}, k1[4], k2[4], k3[4], k4[4], yt[4];
    for (int64_t st = 0; st < nsteps; ++st) {
      double t = t0 + (double)st * h;
      oracle_rhs(f, mass, charge, mu[i], v_ref, t, y, k1);
      for (int c = 0; c < 4; ++c) yt[c] = y[c] + 0.5 * h * k1[c];
      oracle_rhs(f, mass, charge, mu[i], v_ref, t + 0.5 * h, yt, k2);
      for (int c = 0; c < 4; ++c) yt[c] = y[c] + 0.5 * h * k2[c];
      oracle_rhs(f, mass, charge, mu[i], v_ref, t + 0.5 * h, yt, k3);
      for (int c = 0; c < 4; ++c) yt[c] = y[c] + h * k3[c];
      oracle_rhs(f, mass, charge, mu[i], v_ref, t + h, yt, k4);
      for (int c = 0; c < 4; ++c) y[c] += h / 6.0 * (k1[c] + 2.0 * k2[c] + 2.0 * k3[c] + k4[c]);
    }
    y_out[0 * n + i] = y[0]; y_out[1 * n + i] = y[1]; y_out[2 * n + i] = y[2];
    y_out[3 * n + i] = y[3] * v_ref;
  }
}
