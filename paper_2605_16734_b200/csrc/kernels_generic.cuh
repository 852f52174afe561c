// kernels_generic.cuh -- shape-agnostic kernels: one thread per point / particle, tables read from global
// memory in the caller's layout, one sincos per harmonic.  This is the path for fields that do not fit the
// warp kernel's packed layout, the engine of gc_field_eval / gc_pert_eval, and the kernel that the warp
// kernel was first validated against.  Same equations and controller as kernels_warp.cuh.
#pragma once
#include "device_math.cuh"
#include "field.cuh"
#include "kernels_grid.cuh"

namespace gc {

// ---- O2 / O3 point evaluations -------------------------------------------------------------------------
struct Profiles { double G, Gs, I, Is, io, ios; };

__device__ __forceinline__ void interp4(const double* tab, int stride, int i0, const double w[4],
                                        const double dw[4], double& v, double& d) {
  const double t0 = __ldg(tab + (size_t)(i0 + 0) * stride), t1 = __ldg(tab + (size_t)(i0 + 1) * stride);
  const double t2 = __ldg(tab + (size_t)(i0 + 2) * stride), t3 = __ldg(tab + (size_t)(i0 + 3) * stride);
  v = fma(w[3], t3, fma(w[2], t2, fma(w[1], t1, w[0] * t0)));
  d = fma(dw[3], t3, fma(dw[2], t2, fma(dw[1], t1, dw[0] * t0)));
}

// One Fourier series X = sum_k [ xc_k(s) cos(a_k) + xs_k(s) sin(a_k) ], a_k = m_k theta - n_k nfp zeta, with its
// derivatives in s, theta, zeta; either table may be nullptr (NEXT-4: the sin table of B, both tables of K).
// The harmonic list comes in the caller's order, so the trig factors are looked up by (m, n): cos / sin (m theta) and
// cos / sin (n nfp zeta) are built once per call by angle-addition recurrences from ONE sincos each (north_star piece
// 2) into small per-thread tables, and cos(a_k) = c_m C_n + s_m S_n, sin(a_k) = s_m C_n - c_m S_n cost two FMA each
// instead of a 40-instruction sincos per harmonic.  Fields with max m or max |n| above kGenericTrigMax keep one sincos
// per harmonic.
constexpr int kGenericTrigMax = 32;

__device__ inline void eval_series_generic(const FieldDev& f, const double* tabc, const double* tabs, int i0,
                                           const double w[4], const double dw[4], double th, double ze, double out[4],
                                           const double* tabc4 = nullptr, const double* tabs4 = nullptr) {
  const double thr = reduce_2pi(th);
  const double phr = reduce_2pi((double)f.nfp * ze);
  double B = 0.0, Bs = 0.0, Bth = 0.0, Bze = 0.0;
  const bool tables = f.M <= kGenericTrigMax && f.N <= kGenericTrigMax;
  double cm[kGenericTrigMax + 1], sm[kGenericTrigMax + 1], cn[kGenericTrigMax + 1], sn_[kGenericTrigMax + 1];
  if (tables) {
    double s1, c1;
    sincos_poly(thr, s1, c1);
    cm[0] = 1.0; sm[0] = 0.0;
    for (int m = 1; m <= f.M; ++m) {
      cm[m] = fma(cm[m - 1], c1, -sm[m - 1] * s1);
      sm[m] = fma(sm[m - 1], c1, cm[m - 1] * s1);
    }
    sincos_poly(phr, s1, c1);
    cn[0] = 1.0; sn_[0] = 0.0;
    for (int n = 1; n <= f.N; ++n) {
      cn[n] = fma(cn[n - 1], c1, -sn_[n - 1] * s1);
      sn_[n] = fma(sn_[n - 1], c1, cn[n - 1] * s1);
    }
  }
  // four harmonics per pass: one 256-bit load per stencil row and table (rows padded to nhp, field.cuh)
  const bool vec = tables && (!tabc || tabc4) && (!tabs || tabs4);
  const int nloop = vec ? f.nhp : f.nh;
  for (int k0 = 0; k0 < nloop; k0 += vec ? 4 : 1) {
    double bc[4], bcs[4], bsn[4], bss[4];
    if (vec) {
#pragma unroll
      for (int e = 0; e < 4; ++e) bc[e] = bcs[e] = bsn[e] = bss[e] = 0.0;
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        double t[4];
        if (tabc) {
          ldg256(tabc4 + (size_t)(i0 + a) * f.nhp + k0, t[0], t[1], t[2], t[3]);
#pragma unroll
          for (int e = 0; e < 4; ++e) { bc[e] = fma(w[a], t[e], bc[e]); bcs[e] = fma(dw[a], t[e], bcs[e]); }
        }
        if (tabs) {
          ldg256(tabs4 + (size_t)(i0 + a) * f.nhp + k0, t[0], t[1], t[2], t[3]);
#pragma unroll
          for (int e = 0; e < 4; ++e) { bsn[e] = fma(w[a], t[e], bsn[e]); bss[e] = fma(dw[a], t[e], bss[e]); }
        }
      }
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      if (!vec && e > 0) break;
      const int k = k0 + e;
      const int mi = __ldg((vec ? f.xmp : f.xm) + k), ni = __ldg((vec ? f.xnp : f.xn) + k);
      const double m = (double)mi, n = (double)ni;
      double sn, cs;
      if (tables) {
        const int na = ni < 0 ? -ni : ni;
        const double Sn = ni < 0 ? -sn_[na] : sn_[na];              // sin(n phi) is odd in n
        cs = fma(cm[mi], cn[na], sm[mi] * Sn);                      // cos(m theta - n phi)
        sn = fma(sm[mi], cn[na], -cm[mi] * Sn);                     // sin(m theta - n phi)
      } else {
        sincos_poly(fma(m, thr, -n * phr), sn, cs);
      }
      if (tabc) {
        double b, bs;
        if (vec) { b = bc[e]; bs = bcs[e]; }
        else interp4(tabc + k, f.nh, i0, w, dw, b, bs);
        B = fma(b, cs, B);
        Bs = fma(bs, cs, Bs);
        Bth = fma(-m * b, sn, Bth);
        Bze = fma(n * (double)f.nfp * b, sn, Bze);
      }
      if (tabs) {
        double b, bs;
        if (vec) { b = bsn[e]; bs = bss[e]; }
        else interp4(tabs + k, f.nh, i0, w, dw, b, bs);
        B = fma(b, sn, B);
        Bs = fma(bs, sn, Bs);
        Bth = fma(m * b, cs, Bth);
        Bze = fma(-n * (double)f.nfp * b, cs, Bze);
      }
    }
  }
  out[0] = B; out[1] = Bs; out[2] = Bth; out[3] = Bze;
}

__device__ inline void eval_B_generic(const FieldDev& f, int i0, const double w[4], const double dw[4],
                                      double th, double ze, double out[4]) {
  eval_series_generic(f, f.bmnc, f.bmns, i0, w, dw, th, ze, out, f.bmnc4, f.bmns4);
}

// out = Phi, Phi_psi, Phi_th, Phi_ze, al, al_psi, al_th, al_ze, al_t
__device__ inline void eval_pert_generic(const FieldDev& f, int i0, const double w[4], const double dw[4],
                                         const Profiles& p, double th, double ze, double t, double out[9]) {
  double Phi = 0, Phi_s = 0, Phi_th = 0, Phi_ze = 0, al = 0, al_s = 0, al_th = 0, al_ze = 0, al_t = 0;
  const double thr = reduce_2pi(th), zer = reduce_2pi(ze);
  const double GI = p.G + p.io * p.I, GI_s = p.Gs + p.ios * p.I + p.io * p.Is;
  const double invGI = 1.0 / GI, gig = GI_s * invGI;          // one division per evaluation, not one per mode
  for (int k = 0; k < f.nk; ++k) {
    double ph, ph_s;
    interp4(f.phihat + k, f.nk, i0, w, dw, ph, ph_s);
    const double m = (double)__ldg(f.mode_m + k), n = (double)__ldg(f.mode_n + k);
    const double om = __ldg(f.omega + k);
    const double wt = reduce_2pi(om * t);
    double sn, cs;
    sincos_poly(fma(m, thr, fma(-n, zer, wt + __ldg(f.phase + k))), sn, cs);
    // alpha_hat = -Phi_hat (iota m - n) / (omega (G + iota I))    (O3)
    const double inv = __ldg(f.inv_omega + k) * invGI;         // 1 / (omega (G + iota I))
    const double N = fma(p.io, m, -n);
    const double ah = -ph * N * inv;
    const double ah_s = -(ph_s * N + ph * p.ios * m) * inv + ph * N * inv * gig;
    Phi = fma(ph, sn, Phi);
    Phi_s = fma(ph_s, sn, Phi_s);
    Phi_th = fma(m * ph, cs, Phi_th);
    Phi_ze = fma(-n * ph, cs, Phi_ze);
    al = fma(ah, sn, al);
    al_s = fma(ah_s, sn, al_s);
    al_th = fma(m * ah, cs, al_th);
    al_ze = fma(-n * ah, cs, al_ze);
    al_t = fma(om * ah, cs, al_t);
  }
  out[0] = Phi; out[1] = Phi_s * f.inv_psi0; out[2] = Phi_th; out[3] = Phi_ze;
  out[4] = al; out[5] = al_s * f.inv_psi0; out[6] = al_th; out[7] = al_ze; out[8] = al_t;
}

// ---- O4: guiding-centre algebra, shared by both kernels --------------------------------------------------
// fb = B, B_s, B_th, B_ze; pt = perturbation block (all zero for a static field); v = v_par in m/s.
// Returns ds/dt, dtheta/dt, dzeta/dt, d(v_par)/dt.
__device__ __forceinline__ void gc_algebra(double mass, double charge, double mu, double inv_psi0,
                                           double v, const double fb[4], const Profiles& p,
                                           const double pt[9], double dy[4]) {
  const double B = fb[0], B_psi = fb[1] * inv_psi0, B_th = fb[2], B_ze = fb[3];
  const double G = p.G, Gp = p.Gs * inv_psi0, I = p.I, Ip = p.Is * inv_psi0;
  const double Phi_psi = pt[1], Phi_th = pt[2], Phi_ze = pt[3];
  const double al = pt[4], al_psi = pt[5], al_th = pt[6], al_ze = pt[7], al_t = pt[8];
  const double invB = 1.0 / B;
  const double rho_c = mass * v * invB / charge + al;
  const double Fq = (mass * v * v * invB + mu) / charge;
  const double a = 1.0 + rho_c * Ip + al_psi * I;
  const double b = p.io - rho_c * Gp - al_psi * G;
  const double invD = 1.0 / (a * G + b * I);
  const double C = al_th * G - al_ze * I;
  const double h_psi = fma(Fq, B_psi, Phi_psi), h_th = fma(Fq, B_th, Phi_th), h_ze = fma(Fq, B_ze, Phi_ze);
  const double vB = v * B;
  const double Lam = a * B_ze + b * B_th + C * B_psi;
  dy[0] = (I * h_ze - G * h_th + C * vB) * invD * inv_psi0;
  dy[1] = (b * vB + G * h_psi) * invD;
  dy[2] = (a * vB - I * h_psi) * invD;
  const double mvdot = (-mu * B * Lam - charge * B * (a * Phi_ze + b * Phi_th + C * Phi_psi)
                        + mass * v * invB * (B_psi * (I * Phi_ze - G * Phi_th) + Phi_psi * (G * B_th - I * B_ze)))
                           * invD - charge * B * al_t;
  dy[3] = mvdot / mass;
}

// The same with 1 / mass and 1 / charge given (the warp kernel: its right-hand side is one warp's dependent chain,
// where each of the three FP64 divisions by mass and charge costs ~200 cycles of latency; rounding-level difference).
__device__ __forceinline__ void gc_algebra_r(double mass, double charge, double inv_mass, double inv_charge, double mu,
                                             double inv_psi0, double v, const double fb[4], const Profiles& p,
                                             const double pt[9], double dy[4]) {
  const double B = fb[0], B_psi = fb[1] * inv_psi0, B_th = fb[2], B_ze = fb[3];
  const double G = p.G, Gp = p.Gs * inv_psi0, I = p.I, Ip = p.Is * inv_psi0;
  const double Phi_psi = pt[1], Phi_th = pt[2], Phi_ze = pt[3];
  const double al = pt[4], al_psi = pt[5], al_th = pt[6], al_ze = pt[7], al_t = pt[8];
  const double invB = 1.0 / B;
  const double rho_c = mass * v * invB * inv_charge + al;
  const double Fq = (mass * v * v * invB + mu) * inv_charge;
  const double a = 1.0 + rho_c * Ip + al_psi * I;
  const double b = p.io - rho_c * Gp - al_psi * G;
  const double invD = 1.0 / (a * G + b * I);
  const double C = al_th * G - al_ze * I;
  const double h_psi = fma(Fq, B_psi, Phi_psi), h_th = fma(Fq, B_th, Phi_th), h_ze = fma(Fq, B_ze, Phi_ze);
  const double vB = v * B;
  const double Lam = a * B_ze + b * B_th + C * B_psi;
  dy[0] = (I * h_ze - G * h_th + C * vB) * invD * inv_psi0;
  dy[1] = (b * vB + G * h_psi) * invD;
  dy[2] = (a * vB - I * h_psi) * invD;
  const double mvdot = (-mu * B * Lam - charge * B * (a * Phi_ze + b * Phi_th + C * Phi_psi)
                        + mass * v * invB * (B_psi * (I * Phi_ze - G * Phi_th) + Phi_psi * (G * B_th - I * B_ze)))
                           * invD - charge * B * al_t;
  dy[3] = mvdot * inv_mass;
}

// O4 with the covariant radial component K kept (NEXT-4).  The Euler-Lagrange equations of
//   L = q [ rho_c K psidot + (psi + rho_c I) thetadot + (rho_c G - chi) zetadot ] - H,   H = m v^2 / 2 + mu B + q Phi,
// are  sum_j w_ij zdot_j = R_i  (z = psi, theta, zeta, v) with the antisymmetric w_ij = d_i A*_j - d_j A*_i and
// R_i = d_i H / q + d_t A*_i; a 4 x 4 antisymmetric matrix is inverted in closed form through its Pfaffian:
//   w^-1 = [[0, -w34, w24, -w23], [w34, 0, -w14, w13], [-w24, w14, 0, -w12], [w23, -w13, w12, 0]] / Pf,
//   Pf = w12 w34 - w13 w24 + w14 w23.   fk = K, K_s (unused), K_theta, K_zeta.  For K = 0 this is gc_algebra.
__device__ __forceinline__ void gc_algebra_general(double mass, double charge, double mu, double inv_psi0, double v,
                                                   const double fb[4], const double fk[4], const Profiles& p,
                                                   const double pt[9], double dy[4]) {
  const double B = fb[0], B_psi = fb[1] * inv_psi0, B_th = fb[2], B_ze = fb[3];
  const double K = fk[0], K_th = fk[2], K_ze = fk[3];
  const double G = p.G, Gp = p.Gs * inv_psi0, I = p.I, Ip = p.Is * inv_psi0;
  const double al = pt[4], al_t = pt[8];
  const double invB = 1.0 / B, invq = 1.0 / charge;
  const double rv = mass * invB * invq;                    // d rho_c / d v
  const double rho = rv * v, rho_c = rho + al;
  const double r_psi = fma(-rho * invB, B_psi, pt[5]), r_th = fma(-rho * invB, B_th, pt[6]),
               r_ze = fma(-rho * invB, B_ze, pt[7]);
  const double w12 = 1.0 + r_psi * I + rho_c * Ip - r_th * K - rho_c * K_th;
  const double w13 = r_psi * G + rho_c * Gp - p.io - r_ze * K - rho_c * K_ze;
  const double w14 = -rv * K, w23 = r_th * G - r_ze * I, w24 = -rv * I, w34 = -rv * G;
  const double R1 = fma(mu * invq, B_psi, pt[1]) + al_t * K, R2 = fma(mu * invq, B_th, pt[2]) + al_t * I,
               R3 = fma(mu * invq, B_ze, pt[3]) + al_t * G, R4 = mass * v * invq;
  const double invPf = 1.0 / (w12 * w34 - w13 * w24 + w14 * w23);
  dy[0] = (-w34 * R2 + w24 * R3 - w23 * R4) * invPf * inv_psi0;
  dy[1] = (w34 * R1 - w14 * R3 + w13 * R4) * invPf;
  dy[2] = (-w24 * R1 + w14 * R2 - w12 * R4) * invPf;
  dy[3] = (w23 * R1 - w13 * R2 + w12 * R3) * invPf;
}

// y = (s, theta, zeta, u = v_par / v_ref); dy in the same scaled variables.
__device__ inline void rhs_generic(const FieldDev& f, double mass, double charge, double mu, double v_ref,
                                   double inv_v_ref, double t, const double y[4], double dy[4]) {
  int i0;
  double w[4], dw[4], fb[4], pt[9];
  lagrange_weights(f.ns, y[0], i0, w, dw);
  Profiles p;
  interp4(f.G, 1, i0, w, dw, p.G, p.Gs);
  interp4(f.I, 1, i0, w, dw, p.I, p.Is);
  interp4(f.iota, 1, i0, w, dw, p.io, p.ios);
  eval_B_generic(f, i0, w, dw, y[1], y[2], fb);
  if (f.nk > 0) {
    eval_pert_generic(f, i0, w, dw, p, y[1], y[2], t, pt);
  } else {
#pragma unroll
    for (int i = 0; i < 9; ++i) pt[i] = 0.0;
  }
  if (f.kmnc || f.kmns) {
    double fk[4];
    eval_series_generic(f, f.kmnc, f.kmns, i0, w, dw, y[1], y[2], fk, f.kmnc4, f.kmns4);
    gc_algebra_general(mass, charge, mu, f.inv_psi0, y[3] * v_ref, fb, fk, p, pt, dy);
  } else {
    gc_algebra(mass, charge, mu, f.inv_psi0, y[3] * v_ref, fb, p, pt, dy);
  }
  dy[3] *= inv_v_ref;
}

// The same with B from a tricubic interpolant (NEXT-2; KIND 1 Lagrange, 2 Hermite); profiles and perturbation from the
// radial tables as always.
template <int KIND>
__device__ inline void rhs_grid(const FieldDev& f, double mass, double charge, double mu, double v_ref,
                                double inv_v_ref, double t, const double y[4], double dy[4]) {
  int i0;
  double w[4], dw[4], fb[4], pt[9];
  lagrange_weights(f.ns, y[0], i0, w, dw);
  Profiles p;
  interp4(f.G, 1, i0, w, dw, p.G, p.Gs);
  interp4(f.I, 1, i0, w, dw, p.I, p.Is);
  interp4(f.iota, 1, i0, w, dw, p.io, p.ios);
  eval_B_interp<KIND>(f, y[0], y[1], y[2], fb);
  if (f.nk > 0) {
    eval_pert_generic(f, i0, w, dw, p, y[1], y[2], t, pt);
  } else {
#pragma unroll
    for (int i = 0; i < 9; ++i) pt[i] = 0.0;
  }
  gc_algebra(mass, charge, mu, f.inv_psi0, y[3] * v_ref, fb, p, pt, dy);
  dy[3] *= inv_v_ref;
}

// ---- O8: Poincare records from the continuous extension of an accepted step ------------------------------
// r1..r5 are the dense-output coefficients of components s, theta, zeta (index 0..2).
struct Dense3 { double r1[3], r2[3], r3[3], r4[3], r5[3]; };

__device__ __forceinline__ void dense_eval(const Dense3& d, int c, double tau, double& y, double& dy) {
  const double sg = 1.0 - tau;
  const double P4 = fma(sg, d.r5[c], d.r4[c]), dP4 = -d.r5[c];
  const double P3 = fma(tau, P4, d.r3[c]), dP3 = fma(tau, dP4, P4);
  const double P2 = fma(sg, P3, d.r2[c]), dP2 = fma(sg, dP3, -P3);
  y = fma(tau, P2, d.r1[c]);
  dy = fma(tau, dP2, P2);
}

// Called by ONE thread per particle-step.  zeta0/zeta1 are the step's end values of zeta.
__device__ inline void poincare_emit(const Dense3& d, long long id, double t, double h, double zeta0,
                                     double zeta1, double* buf, long long cap, unsigned long long* count) {
  constexpr double kTwoPi = 6.283185307179586476925286766559;
  const double k0 = floor(zeta0 / kTwoPi), k1 = floor(zeta1 / kTwoPi);
  if (k0 == k1) return;
  const double kstep = k1 > k0 ? 1.0 : -1.0;
  const double kfirst = k1 > k0 ? k0 + 1.0 : k0;
  const double klast = k1 > k0 ? k1 : k1 + 1.0;
  for (double kp = kfirst; kstep > 0 ? kp <= klast : kp >= klast; kp += kstep) {
    const double target = kTwoPi * kp;
    double lo = 0.0, hi = 1.0, glo = zeta0 - target, yv, dv;
    for (int it = 0; it < 8; ++it) {
      const double mid = 0.5 * (lo + hi);
      dense_eval(d, 2, mid, yv, dv);
      const double g = yv - target;
      if ((g < 0.0) == (glo < 0.0) && g != 0.0) { lo = mid; glo = g; } else { hi = mid; }
    }
    double tau = 0.5 * (lo + hi);
    const double tol = 1e-12 * fmax(1.0, fabs(target));
    for (int it = 0; it < 20; ++it) {
      dense_eval(d, 2, tau, yv, dv);
      const double g = yv - target;
      if (fabs(g) < tol || dv == 0.0) break;
      tau = fmin(fmax(tau - g / dv, lo), hi);
    }
    const unsigned long long slot = atomicAdd(count, 1ULL);
    if ((long long)slot < cap) {
      double sv, thv;
      dense_eval(d, 0, tau, sv, dv);
      dense_eval(d, 1, tau, thv, dv);
      double thm = fmod(thv, kTwoPi);
      if (thm < 0.0) thm += kTwoPi;
      double* r = buf + slot * 4;
      r[0] = (double)id; r[1] = fma(tau, h, t); r[2] = sv; r[3] = thm;
    }
  }
}

// ---- O9: uniform-time samples of the continuous extension ------------------------------------------------------
__device__ __forceinline__ double sample_time(const TraceDev& p, long long j) {
  return fma((double)j, p.sample_dt, p.sample_t0);          // one FMA on both sides (oracle: sample_time)
}

// First sample index of a particle that starts at t0: first j with tau_j >= t0 (0 .. nsamp).
__device__ __forceinline__ long long first_sample_index(const TraceDev& p, double t0) {
  double g = ceil((t0 - p.sample_t0) / p.sample_dt);
  long long j = g > 0.0 ? (g < (double)p.nsamp ? (long long)g : p.nsamp) : 0;
  while (j > 0 && sample_time(p, j - 1) >= t0) --j;
  while (j < p.nsamp && sample_time(p, j) < t0) ++j;
  return j;
}

// Component c of the continuous extension at tau from y, y_new, h k1, h k7 and h sum d_i k_i.
__device__ __forceinline__ double dense_component(double y, double yn, double hk1, double hk7, double hd, double tau) {
  const double r2 = yn - y, r3 = hk1 - r2, r4 = r2 - hk7 - r3, sg = 1.0 - tau;
  return fma(tau, fma(sg, fma(tau, fma(sg, hd, r4), r3), r2), y);
}

// d/dtau of dense_component.
__device__ __forceinline__ double dense_component_slope(double y, double yn, double hk1, double hk7, double hd,
                                                        double tau) {
  const double r2 = yn - y, r3 = hk1 - r2, r4 = r2 - hk7 - r3, sg = 1.0 - tau;
  const double P4 = fma(sg, hd, r4), dP4 = -hd;
  const double P3 = fma(tau, P4, r3), dP3 = fma(tau, dP4, P4);
  const double P2 = fma(sg, P3, r2), dP2 = fma(sg, dP3, -P3);
  return fma(tau, dP2, P2);
}

// O8b: the bounce section v_par = 0 (u = v_par / v_ref changes sign over the accepted step, or ends on 0).  Called by
// ONE thread per particle-step with y, y_new and h k1, h k7, h sum d_i k_i of the four components.
__device__ __forceinline__ bool bounce_crossed(double u0, double u1) {
  return (u0 < 0.0 && u1 >= 0.0) || (u0 > 0.0 && u1 <= 0.0);
}
__device__ inline void bounce_emit(const double (&y)[4], const double (&yn)[4], const double (&hk1)[4],
                                   const double (&hk7)[4], const double (&hd)[4], long long id, double t, double h,
                                   double* buf, long long cap, unsigned long long* count) {
  constexpr double kTwoPi = 6.283185307179586476925286766559;
  double lo = 0.0, hi = 1.0, glo = y[3];
  for (int it = 0; it < 8; ++it) {
    const double mid = 0.5 * (lo + hi);
    const double g = dense_component(y[3], yn[3], hk1[3], hk7[3], hd[3], mid);
    if ((g < 0.0) == (glo < 0.0) && g != 0.0) { lo = mid; glo = g; } else { hi = mid; }
  }
  double tau = 0.5 * (lo + hi);
  for (int it = 0; it < 20; ++it) {
    const double g = dense_component(y[3], yn[3], hk1[3], hk7[3], hd[3], tau);
    const double dv = dense_component_slope(y[3], yn[3], hk1[3], hk7[3], hd[3], tau);
    if (fabs(g) < 1e-12 || dv == 0.0) break;
    tau = fmin(fmax(tau - g / dv, lo), hi);
  }
  const unsigned long long slot = atomicAdd(count, 1ULL);
  if ((long long)slot < cap) {
    const double sv = dense_component(y[0], yn[0], hk1[0], hk7[0], hd[0], tau);
    const double thv = dense_component(y[1], yn[1], hk1[1], hk7[1], hd[1], tau);
    double thm = fmod(thv, kTwoPi);
    if (thm < 0.0) thm += kTwoPi;
    double* r = buf + slot * 4;
    r[0] = (double)id; r[1] = fma(tau, h, t); r[2] = sv; r[3] = thm;
  }
}

// O7b: root of s(tau) = s_loss on the continuous extension of component 0 (s < s_loss at tau = 0, >= at tau = 1).
__device__ inline double loss_root(double y0, double yn0, double hk1, double hk7, double hd, double s_loss) {
  double lo = 0.0, hi = 1.0;
  for (int it = 0; it < 8; ++it) {
    const double mid = 0.5 * (lo + hi);
    if (dense_component(y0, yn0, hk1, hk7, hd, mid) < s_loss) lo = mid; else hi = mid;
  }
  double tau = 0.5 * (lo + hi);
  for (int it = 0; it < 20; ++it) {
    const double g = dense_component(y0, yn0, hk1, hk7, hd, tau) - s_loss;
    const double dv = dense_component_slope(y0, yn0, hk1, hk7, hd, tau);
    if (fabs(g) < 1e-14 || dv == 0.0) break;
    tau = fmin(fmax(tau - g / dv, lo), hi);
  }
  return tau;
}

// ---- A17: P_zeta = q ((rho + alpha) G - chi) at n states and times ----------------------------------------------
__global__ void pzeta_eval_kernel(FieldDev f, double mass, double charge, long long n, const double* y,
                                  const double* t, const double* chi_nodes, double* out) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double s = y[i], th = y[n + i], ze = y[2 * n + i], v = y[3 * n + i];
  int i0;
  double w[4], dw[4], fb[4], pt[9];
  lagrange_weights(f.ns, s, i0, w, dw);
  Profiles p;
  interp4(f.G, 1, i0, w, dw, p.G, p.Gs);
  interp4(f.I, 1, i0, w, dw, p.I, p.Is);
  interp4(f.iota, 1, i0, w, dw, p.io, p.ios);
  if (f.grid) eval_B_interp_rt(f, s, th, ze, fb);
  else eval_B_generic(f, i0, w, dw, th, ze, fb);
  double al = 0.0;
  if (f.nk > 0) {
    eval_pert_generic(f, i0, w, dw, p, th, ze, t ? t[i] : 0.0, pt);
    al = pt[4];
  }
  double chi, dchi;
  interp4(chi_nodes, 1, i0, w, dw, chi, dchi);
  const double rho = mass * v / (charge * fb[0]);
  out[i] = charge * ((rho + al) * p.G - chi);
}

// ---- A25: weighted Birkhoff average of the two halves of each series, digit accuracy ---------------------------------
__global__ void birkhoff_kernel(long long n, long long nsamp, const double* series, long long j_first,
                                const int* sample_end, double* out) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  long long end = sample_end ? (long long)sample_end[i] : nsamp;
  if (end > nsamp) end = nsamp;
  const long long N = (end - j_first) / 2;
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  if (j_first < 0 || N < 2) { out[i] = nan; out[n + i] = nan; out[2 * n + i] = nan; return; }
  double wb[2];
  for (int half = 0; half < 2; ++half) {
    double sw = 0.0, swf = 0.0;
    const double* fcol = series + (j_first + half * N) * n + i;
    for (long long k = 0; k < N; ++k) {
      const double x = (double)(k + 1) / (double)(N + 1);
      const double w = exp(-1.0 / (x * (1.0 - x)));
      sw += w;
      swf = fma(w, fcol[k * n], swf);
    }
    wb[half] = swf / sw;
  }
  const double d = fabs(wb[0] - wb[1]), scale = fmax(fabs(wb[0]), fabs(wb[1]));
  out[i] = wb[0];
  out[n + i] = wb[1];
  out[2 * n + i] = (d == 0.0 || scale == 0.0) ? 16.0 : fmin(16.0, -log10(d / scale));
}

// ---- A30: orbit classification, characteristic frequencies, J_par of n series of uniform-time samples -----------------
// samples [4][nsamp][n] (gc_trace_sampled / gc_trace_symplectic layout); out [7][n] = class (0 passing, 1 trapped),
// reversals of v_par, omega_theta, omega_zeta, omega_bounce, mean J_par over the full bounce periods, (max - min) / mean.
__global__ void orbit_diag_kernel(long long n, long long nsamp, const double* samples, long long j_first,
                                  const int* sample_end, double dt, double mass, double* out) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  long long end = sample_end ? (long long)sample_end[i] : nsamp;
  if (end > nsamp) end = nsamp;
  const long long c = end - j_first;
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  if (j_first < 0 || c < 2) {
    out[i] = nan; out[n + i] = 0.0;
#pragma unroll
    for (int q = 2; q < 7; ++q) out[q * n + i] = nan;
    return;
  }
  const double* th = samples + (1 * nsamp + j_first) * n + i;
  const double* ze = samples + (2 * nsamp + j_first) * n + i;
  const double* vp = samples + (3 * nsamp + j_first) * n + i;
  // pass 1: count the reversals and find the first one
  long long R = 0;
  double v0 = vp[0];
  for (long long j = 0; j + 1 < c; ++j) {
    const double v1 = vp[(j + 1) * n];
    if ((v0 < 0.0) != (v1 < 0.0)) ++R;
    v0 = v1;
  }
  const long long P = R >= 3 ? (R - 1) / 2 : 0;
  double omega_b = 0.0, jmean = nan, jvar = nan;
  if (P > 0) {
    // pass 2: walk the reversals 0 .. 2 P; between reversal 2 p and 2 p + 2 integrate m v^2 dt by the trapezoid rule
    long long r = -1;                    // index of the last reversal seen
    double tau0 = 0.0, tau_last = 0.0, acc = 0.0, jsum = 0.0, jmin = 0.0, jmax = 0.0;
    v0 = vp[0];
    for (long long j = 0; j + 1 < c && r < 2 * P; ++j) {
      const double v1 = vp[(j + 1) * n];
      if ((v0 < 0.0) != (v1 < 0.0)) {
        const double tau = (double)j * dt + dt * v0 / (v0 - v1);
        ++r;
        if (r == 0) {
          tau0 = tau;
          acc = 0.5 * v1 * v1 * ((double)(j + 1) * dt - tau);                  // reversal -> first sample of the period
        } else if (r & 1) {
          acc += 0.5 * (v0 * v0 + v1 * v1) * dt;                                // the reversal in the middle of a period
        } else {
          acc += 0.5 * v0 * v0 * (tau - (double)j * dt);                        // last sample of the period -> reversal
          const double J = mass * acc;
          jsum += J;
          jmin = r == 2 ? J : fmin(jmin, J);
          jmax = r == 2 ? J : fmax(jmax, J);
          acc = 0.5 * v1 * v1 * ((double)(j + 1) * dt - tau);
        }
        tau_last = tau;
      } else if (r >= 0) {
        acc += 0.5 * (v0 * v0 + v1 * v1) * dt;
      }
      v0 = v1;
    }
    omega_b = 6.283185307179586476925286766559 * (double)P / (tau_last - tau0);
    jmean = jsum / (double)P;
    jvar = (jmax - jmin) / jmean;
  }
  const double T = (double)(c - 1) * dt;
  out[i] = R >= 1 ? 1.0 : 0.0;
  out[n + i] = (double)R;
  out[2 * n + i] = (th[(c - 1) * n] - th[0]) / T;
  out[3 * n + i] = (ze[(c - 1) * n] - ze[0]) / T;
  out[4 * n + i] = omega_b;
  out[5 * n + i] = jmean;
  out[6 * n + i] = jvar;
}

__global__ void field_eval_kernel(FieldDev f, long long n, const double* s, const double* th, const double* ze,
                                  double* B, double* dB) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  int i0;
  double w[4], dw[4], out[4];
  if (f.grid) {
    eval_B_interp_rt(f, s[i], th[i], ze[i], out);          // NEXT-2: the field is the interpolant
  } else {
    lagrange_weights(f.ns, s[i], i0, w, dw);
    eval_B_generic(f, i0, w, dw, th[i], ze[i], out);
  }
  B[i] = out[0];
  if (dB) { dB[i] = out[1]; dB[n + i] = out[2]; dB[2 * n + i] = out[3]; }
}

// NEXT-2 setup, step 1: node values of B (direct sum O2), plain[ngs][nth][nze].  One thread per node.
__global__ void grid_build_kernel(FieldDev f, int ngs, int nth, int nze, double* plain) {
  constexpr double kTwoPi = 6.283185307179586476925286766559;
  const long long total = (long long)ngs * nth * nze;
  const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (e >= total) return;
  const int k = (int)(e % nze);
  const int j = (int)((e / nze) % nth);
  const int i = (int)(e / ((long long)nze * nth));
  const double s = (double)i / (double)(ngs - 1);
  const double th = kTwoPi * (double)j / (double)nth;
  const double ze = kTwoPi * (double)k / ((double)nze * (double)f.nfp);
  int i0;
  double w[4], dw[4], out[4];
  lagrange_weights(f.ns, s, i0, w, dw);
  eval_B_generic(f, i0, w, dw, th, ze, out);
  plain[e] = out[0];
}

// Step 2: the gather layout of kernels_grid.cuh, grid[ngs][nth + 3][nze][4]: entry (i, jp, k) = nodes k .. k+3 (mod
// nze) of row (i, jp mod nth).  One thread per entry.
__global__ void grid_pack_kernel(int ngs, int nth, int nze, const double* plain, double* grid) {
  const long long total = (long long)ngs * (nth + 3) * nze;
  const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (e >= total) return;
  const int k = (int)(e % nze);
  const int jp = (int)((e / nze) % (nth + 3));
  const int i = (int)(e / ((long long)nze * (nth + 3)));
  const double* row = plain + ((long long)i * nth + jp % nth) * nze;
#pragma unroll
  for (int c = 0; c < 4; ++c) grid[e * 4 + c] = row[(k + c) % nze];
}

// Setup of the Hermite variant (A31): per node the direct sum and its seven first and mixed derivatives, term by term,
// pre-multiplied by the cell widths of the differentiated directions, in the layout of field.cuh:
// grid[ngs][nth + 1][nze + 1][8] = (f, f_ze, f_th, f_th_ze, f_s, f_s_ze, f_s_th, f_s_th_ze).  One thread per entry.
__global__ void grid8_build_kernel(FieldDev f, int ngs, int nth, int nze, double* grid) {
  constexpr double kTwoPi = 6.283185307179586476925286766559;
  const long long total = (long long)ngs * (nth + 1) * (nze + 1);
  const long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (e >= total) return;
  const int kp = (int)(e % (nze + 1));
  const int jp = (int)((e / (nze + 1)) % (nth + 1));
  const int i = (int)(e / ((long long)(nze + 1) * (nth + 1)));
  const int j = jp % nth, k = kp % nze;
  const double s = (double)i / (double)(ngs - 1);
  const double th = kTwoPi * (double)j / (double)nth;
  const double ze = kTwoPi * (double)k / ((double)nze * (double)f.nfp);
  const double ds = 1.0 / (double)(ngs - 1), dth = kTwoPi / (double)nth, dze = kTwoPi / ((double)nze * (double)f.nfp);
  int i0;
  double w[4], dw[4];
  lagrange_weights(f.ns, s, i0, w, dw);
  const double thr = reduce_2pi(th), phr = reduce_2pi((double)f.nfp * ze);
  double o[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};     // f, f_s, f_th, f_ze, f_s_th, f_s_ze, f_th_ze, f_s_th_ze
  for (int h = 0; h < f.nh; ++h) {
    const double m = (double)__ldg(f.xm + h), nn = (double)__ldg(f.xn + h) * (double)f.nfp;
    double sn, cs;
    sincos_poly(fma(m, thr, -(double)__ldg(f.xn + h) * phr), sn, cs);
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
      const double* tab = pass == 0 ? f.bmnc : f.bmns;
      if (!tab) continue;
      double b, bs;
      interp4(tab + h, f.nh, i0, w, dw, b, bs);
      const double v = pass == 0 ? cs : sn;
      const double vth = pass == 0 ? -m * sn : m * cs;
      const double vze = pass == 0 ? nn * sn : -nn * cs;
      const double vtz = pass == 0 ? m * nn * cs : m * nn * sn;
      o[0] = fma(b, v, o[0]);     o[1] = fma(bs, v, o[1]);
      o[2] = fma(b, vth, o[2]);   o[3] = fma(b, vze, o[3]);
      o[4] = fma(bs, vth, o[4]);  o[5] = fma(bs, vze, o[5]);
      o[6] = fma(b, vtz, o[6]);   o[7] = fma(bs, vtz, o[7]);
    }
  }
  double* g = grid + e * 8;
  g[0] = o[0];            g[1] = o[3] * dze;        g[2] = o[2] * dth;       g[3] = o[6] * dth * dze;
  g[4] = o[1] * ds;       g[5] = o[5] * ds * dze;   g[6] = o[4] * ds * dth;  g[7] = o[7] * ds * dth * dze;
}

__global__ void kcov_eval_kernel(FieldDev f, long long n, const double* s, const double* th, const double* ze,
                                 double* K, double* dK) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  int i0;
  double w[4], dw[4], out[4] = {0.0, 0.0, 0.0, 0.0};
  lagrange_weights(f.ns, s[i], i0, w, dw);
  if (f.kmnc || f.kmns) eval_series_generic(f, f.kmnc, f.kmns, i0, w, dw, th[i], ze[i], out, f.kmnc4, f.kmns4);
  K[i] = out[0];
  if (dK) { dK[i] = out[1]; dK[n + i] = out[2]; dK[2 * n + i] = out[3]; }
}

__global__ void pert_eval_kernel(FieldDev f, long long n, const double* s, const double* th, const double* ze,
                                 double t, double* out) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  int i0;
  double w[4], dw[4], pt[9];
  lagrange_weights(f.ns, s[i], i0, w, dw);
  Profiles p;
  interp4(f.G, 1, i0, w, dw, p.G, p.Gs);
  interp4(f.I, 1, i0, w, dw, p.I, p.Is);
  interp4(f.iota, 1, i0, w, dw, p.io, p.ios);
  if (f.nk > 0) {
    eval_pert_generic(f, i0, w, dw, p, th[i], ze[i], t, pt);
  } else {
    for (int j = 0; j < 9; ++j) pt[j] = 0.0;
  }
  for (int j = 0; j < 9; ++j) out[j * n + i] = pt[j];
}

__global__ void rhs_eval_generic_kernel(FieldDev f, double mass, double charge, double t, long long n,
                                        const double* y, const double* mu, double* dydt) {
  const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double yy[4] = {y[i], y[n + i], y[2 * n + i], y[3 * n + i]};
  double dy[4];
  if (f.grid && f.grid_kind == 2) rhs_grid<2>(f, mass, charge, mu[i], 1.0, 1.0, t, yy, dy);
  else if (f.grid) rhs_grid<1>(f, mass, charge, mu[i], 1.0, 1.0, t, yy, dy);
  else rhs_generic(f, mass, charge, mu[i], 1.0, 1.0, t, yy, dy);
  for (int c = 0; c < 4; ++c) dydt[c * n + i] = dy[c];
}

}  // namespace gc
