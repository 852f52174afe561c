// kernels_symplectic.cuh -- NEXT-3 of SURVEY.md section 8(f): the symplectic explicit-implicit Euler integrator for
// non-canonical guiding-centre orbits ("uses the explicit-implicit Euler scheme of (Albert et al.,
// 2020)"; Fig. 1 left; reading A28 of DESIGN.md).  Static fields with K = 0.
//
// The guiding-centre Lagrangian of O4 without perturbation, L = q (psi + rho I) thetadot + q (rho G - chi) zetadot - H,
// has the canonical momenta p_theta = q (psi0 s + rho I), p_zeta = q (rho G - chi); the state carried is
// z = (s, theta, zeta, p_zeta) and rho(s, p_zeta) = (p_zeta / q + chi(s)) / G(s), H = (q rho B)^2 / (2 m) + mu B.
// One step of size h (symplectic Euler: implicit in the momenta, explicit in the angles):
//     F1 = p_theta(s', p_zeta') - p_theta(s, p_zeta) + h dH/dtheta = 0
//     F2 = p_zeta' - p_zeta + h dH/dzeta = 0                         derivatives at (s', theta, zeta, p_zeta')
//     theta' = theta + h (dH/ds) / (dp_theta/ds)
//     zeta'  = zeta  + h [dH/dp_zeta - (dH/ds) (dp_theta/dp_zeta) / (dp_theta/ds)]
// The 2 x 2 system is solved by a quasi-Newton iteration whose Jacobian is the h = 0 part of the exact one,
// [[dp_theta/ds, dp_theta/dp_zeta], [0, 1]]: every iteration costs ONE evaluation of B and its derivatives (no second
// derivatives of the field), the error shrinks by h |d(dH/dtheta)/ds| / (dp_theta/ds) ~ 1e-3 per iteration, it starts
// from the linear extrapolation of the previous step, and the
// iteration stops when the update of (s, p_zeta / (q psi0)) is below newton_tol max(1, |x|) -- the root the oracle's
// Newton iteration converges to.  The partial derivatives of the last evaluation (within newton_tol of the root) feed
// the explicit half.  One lane per particle; every particle takes the same number of steps, so there is no queue.
#pragma once
#include "kernels_generic.cuh"

namespace gc {

struct SymplecticDev {
  double mass, charge, t0, dt, s_loss, s_min, tol;
  long long nsteps, n, sample_stride, nsamp;
  int max_iter, resume;
  const double *s0, *th0, *ze0, *vpar0, *mu, *chi;
  double *y_out, *t_out;
  int *status, *n_steps, *n_iter;
  double* samples;
  int* sample_end;
};

struct SymPoint {          // everything of one evaluation at (s, theta, zeta, p_zeta)
  double B, Bs, Bth, Bze, G, Gs, I, Is, rho, rho_s, pth, D, dpth_dpz;
};

template <int GRID>
__device__ __forceinline__ void sym_eval(const FieldDev& f, const double* chi_nodes, double q, double s, double th,
                                         double ze, double pz, bool with_field, SymPoint& e) {
  int i0;
  double w[4], dw[4], chi, chi_s;
  lagrange_weights(f.ns, s, i0, w, dw);
  interp4(f.G, 1, i0, w, dw, e.G, e.Gs);
  interp4(f.I, 1, i0, w, dw, e.I, e.Is);
  interp4(chi_nodes, 1, i0, w, dw, chi, chi_s);
  const double invG = 1.0 / e.G;
  e.rho = (pz / q + chi) * invG;
  e.rho_s = (chi_s - e.rho * e.Gs) * invG;
  e.pth = q * fma(e.rho, e.I, f.psi0 * s);
  e.D = q * (f.psi0 + e.rho_s * e.I + e.rho * e.Is);
  e.dpth_dpz = e.I * invG;
  if (with_field) {
    double fb[4];
    if (GRID) eval_B_interp<GRID>(f, s, th, ze, fb);
    else eval_B_generic(f, i0, w, dw, th, ze, fb);
    e.B = fb[0]; e.Bs = fb[1]; e.Bth = fb[2]; e.Bze = fb[3];
  }
}

template <int GRID>
__global__ void __launch_bounds__(128) trace_symplectic_kernel(FieldDev f, SymplecticDev p) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < p.n;
       i += (long long)gridDim.x * blockDim.x) {
    if (p.resume && p.status[i] != 0) continue;
    const double q = p.charge, m = p.mass, mu = p.mu[i], unit = q * f.psi0, inv_unit = 1.0 / unit;
    double s = p.s0[i], th = p.th0[i], ze = p.ze0[i], vpar = p.vpar0[i];
    SymPoint e;
    // p_zeta = q (rho G - chi), rho = m v_par / (q B)   (A17)
    double pz;
    {
      int i0;
      double w[4], dw[4], fb[4], G, Gs, chi, chi_s;
      lagrange_weights(f.ns, s, i0, w, dw);
      if (GRID) eval_B_interp<GRID>(f, s, th, ze, fb);
      else eval_B_generic(f, i0, w, dw, th, ze, fb);
      interp4(f.G, 1, i0, w, dw, G, Gs);
      interp4(p.chi, 1, i0, w, dw, chi, chi_s);
      pz = q * (m * vpar / (q * fb[0]) * G - chi);
    }
    int st = 0, steps = 0, iters = 0;
    long long js = 0;
    if (!finite4(s, th, ze, pz)) st = GC_ST_NONFINITE_;
    if (p.nsamp > 0 && st == 0 && !p.resume) {                // sample 0 is the initial state
      p.samples[(0 * p.nsamp + 0) * p.n + i] = s;  p.samples[(1 * p.nsamp + 0) * p.n + i] = th;
      p.samples[(2 * p.nsamp + 0) * p.n + i] = ze; p.samples[(3 * p.nsamp + 0) * p.n + i] = vpar;
      js = 1;
    } else if (p.nsamp > 0 && p.resume) {
      js = p.sample_end[i];
    }
    sym_eval<GRID>(f, p.chi, q, s, th, ze, pz, false, e);
    double pth_old = e.pth;
    double ds_prev = 0.0, dx1_prev = 0.0;                      // increments of the last step: the predictor
    for (long long k = 0; k < p.nsteps && st == 0; ++k) {
      const double pz_old = pz;
      // start the iteration from the linear extrapolation of the last step (error O(h^2) instead of O(h): one to two
      // iterations fewer; the root it converges to is the same)
      double x0 = s + ds_prev, x1 = pz * inv_unit + dx1_prev;
      bool ok = false;
      int it = 0;
      double H_s = 0.0, H_pz = 0.0;
      while (it < p.max_iter) {
        ++it;
        sym_eval<GRID>(f, p.chi, q, x0, th, ze, x1 * unit, true, e);
        const double qr = q * e.rho;
        const double dHdB = fma(qr * qr / m, e.B, mu);          // dH/dB = q^2 rho^2 B / m + mu
        const double F1 = e.pth - pth_old + p.dt * dHdB * e.Bth;
        const double F2 = fma(x1, unit, -pz_old) + p.dt * dHdB * e.Bze;
        const double dpz = -F2;
        const double ds = -(F1 + e.dpth_dpz * dpz) / e.D;
        const double dx1 = dpz * inv_unit;
        H_s = qr * q * e.rho_s * e.B * e.B / m + dHdB * e.Bs;
        H_pz = qr * e.B * e.B / (m * e.G);
        if (!isfinite(ds) || !isfinite(dx1)) break;
        x0 += ds; x1 += dx1;
        if (fabs(ds) <= p.tol * fmax(1.0, fabs(x0)) && fabs(dx1) <= p.tol * fmax(1.0, fabs(x1))) { ok = true; break; }
      }
      iters += it;
      if (!ok) { st = GC_ST_NONFINITE_; break; }
      // explicit half with the partial derivatives of the last evaluation (within tol of the root)
      const double th_new = fma(p.dt, H_s / e.D, th);
      const double ze_new = fma(p.dt, H_pz - H_s * e.dpth_dpz / e.D, ze);
      // a step that ends on a non-finite value is not committed: the state before it is reported (gcorbit.h), as
      // trace_mma_symplectic_kernel does, so the result does not depend on which engine the ensemble size selects
      if (!finite4(x0, th_new, ze_new, x1 * unit)) { st = GC_ST_NONFINITE_; break; }
      th = th_new;
      ze = ze_new;
      ds_prev = x0 - s;
      dx1_prev = x1 - pz * inv_unit;
      s = x0;
      pz = x1 * unit;
      ++steps;
      sym_eval<GRID>(f, p.chi, q, s, th, ze, pz, false, e);     // profiles at the new point: p_theta of the next step
      pth_old = e.pth;
      if (p.nsamp > 0 && js < p.nsamp && (k + 1) % p.sample_stride == 0) {
        // v_par = q rho B / m at the NEW point needs B there
        int i0;
        double w[4], dw[4], fb[4];
        lagrange_weights(f.ns, s, i0, w, dw);
        if (GRID) eval_B_interp<GRID>(f, s, th, ze, fb);
        else eval_B_generic(f, i0, w, dw, th, ze, fb);
        p.samples[(0 * p.nsamp + js) * p.n + i] = s;  p.samples[(1 * p.nsamp + js) * p.n + i] = th;
        p.samples[(2 * p.nsamp + js) * p.n + i] = ze; p.samples[(3 * p.nsamp + js) * p.n + i] = q * e.rho * fb[0] / m;
        ++js;
      }
      if (s >= p.s_loss) st = 1;
      else if (s <= p.s_min) st = 2;
    }
    if (steps > 0) {
      int i0;
      double w[4], dw[4], fb[4];
      sym_eval<GRID>(f, p.chi, q, s, th, ze, pz, false, e);     // rho at the reported state (a failed step moved e)
      lagrange_weights(f.ns, s, i0, w, dw);
      if (GRID) eval_B_interp<GRID>(f, s, th, ze, fb);
      else eval_B_generic(f, i0, w, dw, th, ze, fb);
      vpar = q * e.rho * fb[0] / m;
    }
    p.y_out[0 * p.n + i] = s; p.y_out[1 * p.n + i] = th; p.y_out[2 * p.n + i] = ze; p.y_out[3 * p.n + i] = vpar;
    p.t_out[i] = __dadd_rn(p.t0, __dmul_rn((double)steps, p.dt));   // as the oracle: one product, one sum
    p.status[i] = st;
    if (p.n_steps) p.n_steps[i] = (p.resume ? p.n_steps[i] : 0) + steps;
    if (p.n_iter) p.n_iter[i] = (p.resume ? p.n_iter[i] : 0) + iters;
    if (p.nsamp > 0) p.sample_end[i] = (int)js;
  }
}

}  // namespace gc
