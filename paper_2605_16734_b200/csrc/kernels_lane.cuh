// kernels_lane.cuh -- one lane per particle with an atomic particle queue: the trace kernel of the 3-D interpolant
// field (NEXT-2, kernels_grid.cuh) and of any field that fits none of the packed layouts (GC_KERNEL_GENERIC).
//
// A persistent grid; every lane holds one particle and all lanes of a warp run the same Dormand-Prince attempt in
// lock step (the attempt is the same instruction sequence for every particle).  Step counts differ by a factor of
// two to three between particles (passing against trapped), so a lane whose particle stops takes the
// next one from a global atomic counter straight away (one warp-aggregated atomicAdd per refill round) instead of
// idling until the slowest particle of its warp ends (north_star piece 3).  A particle's result
// does not depend on which lane ran it.  Same equations and controller as every other kernel.
#pragma once
#include "kernels_generic.cuh"

namespace gc {

constexpr int kLaneThreads = 128;
#ifndef GC_LANE_MIN_BLOCKS
#define GC_LANE_MIN_BLOCKS 2
#endif

// O4 at one state: GRID = 0: direct harmonic sum from the caller's tables (rhs_generic); GRID = 1 / 2: B and its
// derivatives from the tricubic Lagrange / Hermite interpolant, profiles and perturbation from the radial tables.
template <int GRID>
__device__ __forceinline__ void rhs_lane(const FieldDev& f, double mass, double charge, double mu, double v_ref,
                                         double inv_v_ref, double t, const double y[4], double dy[4]) {
  if (GRID == 0) rhs_generic(f, mass, charge, mu, v_ref, inv_v_ref, t, y, dy);
  else rhs_grid<GRID>(f, mass, charge, mu, v_ref, inv_v_ref, t, y, dy);
}

// Dormand-Prince coefficients by stage for the stage loop: row r holds a_{r+2, 1..6} (O5); c_2 .. c_7.
__constant__ double kDpA[6][6] = {
    {dp::a21, 0.0, 0.0, 0.0, 0.0, 0.0},
    {dp::a31, dp::a32, 0.0, 0.0, 0.0, 0.0},
    {dp::a41, dp::a42, dp::a43, 0.0, 0.0, 0.0},
    {dp::a51, dp::a52, dp::a53, dp::a54, 0.0, 0.0},
    {dp::a61, dp::a62, dp::a63, dp::a64, dp::a65, 0.0},
    {dp::a71, 0.0, dp::a73, dp::a74, dp::a75, dp::a76}};
__constant__ double kDpC[6] = {dp::c2, dp::c3, dp::c4, dp::c5, 1.0, 1.0};

constexpr int kLaneSmemBytes = 7 * 4 * kLaneThreads * (int)sizeof(double);

// The seven stage derivatives of a lane live in shared memory, kbuf[7][4][kLaneThreads] (conflict-free: consecutive
// lanes, consecutive doubles): the stages then run as a LOOP around one copy of the right-hand side, which keeps the
// hot loop inside the instruction cache (seven inlined copies were 175 KB of code and the warps stalled on
// instruction fetch) and frees 56 registers per lane for occupancy.
#define GC_K(j, c) kbuf[((j) * 4 + (c)) * kLaneThreads + threadIdx.x]

__device__ __forceinline__ double dense_hd(const double* kbuf, int c, double h) {
  return h * fma(dp::d7, GC_K(6, c), fma(dp::d6, GC_K(5, c), fma(dp::d5, GC_K(4, c),
                 fma(dp::d4, GC_K(3, c), fma(dp::d3, GC_K(2, c), dp::d1 * GC_K(0, c))))));
}

template <int GRID>
__global__ void __launch_bounds__(kLaneThreads, GC_LANE_MIN_BLOCKS) trace_lane_kernel(FieldDev f, TraceDev p) {
  extern __shared__ double kbuf[];
  constexpr unsigned kFull = 0xffffffffu;
  const unsigned lane = threadIdx.x & 31u;
  long long i = -1;                       // the particle this lane holds; -1 = none
  bool drained = false;                   // the queue has no particle left for this lane
  double mu = 0.0, t = 0.0, h = 0.0, y[4], yn[4], ys[4], dy[4];
  long long attempts = 0, jn = 0;
  int n_acc = 0, n_rej = 0, n_forced = 0, st = -1;
  bool prev_rejected = false;
#pragma unroll
  for (int c = 0; c < 4; ++c) y[c] = yn[c] = 0.0;
  for (;;) {
    // ---- refill: lanes without a particle take the next indices of the queue -------------------------------------
    const bool want = i < 0 && !drained;
    const unsigned m = __ballot_sync(kFull, want);
    if (m != 0u) {
      const int leader = __ffs(m) - 1;
      unsigned long long base = 0;
      if ((int)lane == leader) base = atomicAdd(p.work_counter, (unsigned long long)__popc(m));
      base = __shfl_sync(kFull, base, leader);
      if (want) {
        const long long idx = (long long)base + __popc(m & ((1u << lane) - 1u));
        if (idx >= p.n) {
          drained = true;
        } else if (!(p.resume && p.status[idx] != 0)) {      // else: finished in an earlier segment, ask again
          i = idx;
          mu = p.mu[i];
          y[0] = p.s0[i]; y[1] = p.th0[i]; y[2] = p.ze0[i]; y[3] = p.vpar0[i] * p.inv_v_ref;
          t = p.t0;
          h = (p.h_inout && p.h_inout[i] > 0.0) ? p.h_inout[i] : p.h0;
          if (h < p.h_min) h = p.h_min;
          attempts = 0; n_acc = n_rej = n_forced = 0; st = -1; prev_rejected = false; jn = 0;
          if (p.nsamp > 0) {
            jn = first_sample_index(p, t);
            if (jn < p.nsamp && sample_time(p, jn) == t) {       // a sample on t0 is the initial state
#pragma unroll
              for (int c = 0; c < 4; ++c)
                p.samples[((long long)c * p.nsamp + jn) * p.n + i] = c == 3 ? p.vpar0[i] : y[c];
              ++jn;
            }
          }
          rhs_lane<GRID>(f, p.mass, p.charge, mu, p.v_ref, p.inv_v_ref, t, y, dy);
#pragma unroll
          for (int c = 0; c < 4; ++c) GC_K(0, c) = dy[c];
          if (!finite4(y[0], y[1], y[2], y[3]) || !finite4(dy[0], dy[1], dy[2], dy[3])) st = GC_ST_NONFINITE_;
          else if (!(t < p.t_max)) st = 0;
        }
      }
    }
    if (__all_sync(kFull, i < 0 && drained)) break;

    // ---- one attempted step (O5, O6) --------------------------------------------------------------------------------
    if (i >= 0 && st < 0) {
      double h_try = h;
      bool clipped = false;
      if (t + h_try >= p.t_max) { h_try = p.t_max - t; clipped = true; }
      if (!(t + h_try > t)) {
        st = GC_ST_NONFINITE_;                                 // A23: step underflow
      } else {
        const bool forced = prev_rejected && p.h_min > 0.0 && h == p.h_min;
#pragma unroll 1
        for (int sg = 1; sg <= 6; ++sg) {                      // stages 2 .. 7 (the 7th is the FSAL evaluation at y_new)
          double acc[4] = {0.0, 0.0, 0.0, 0.0};
          for (int j = sg - 1; j >= 0; --j) {
            const double a = kDpA[sg - 1][j];
#pragma unroll
            for (int c = 0; c < 4; ++c) acc[c] = fma(a, GC_K(j, c), acc[c]);
          }
#pragma unroll
          for (int c = 0; c < 4; ++c) ys[c] = fma(h_try, acc[c], y[c]);
          const double tt = sg >= 5 ? t + h_try : fma(kDpC[sg - 1], h_try, t);
          rhs_lane<GRID>(f, p.mass, p.charge, mu, p.v_ref, p.inv_v_ref, tt, ys, dy);
#pragma unroll
          for (int c = 0; c < 4; ++c) GC_K(sg, c) = dy[c];
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) yn[c] = ys[c];             // the 5th-order solution is the last stage point
        ++attempts;
        double acc = 0.0;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const double delta = h_try * fma(dp::e7, GC_K(6, c), fma(dp::e6, GC_K(5, c), fma(dp::e5, GC_K(4, c),
                                   fma(dp::e4, GC_K(3, c), fma(dp::e3, GC_K(2, c), dp::e1 * GC_K(0, c))))));
          const double sk = fma(p.rtol, fmax(fabs(y[c]), fabs(yn[c])), p.atol);
          const double r = delta / sk;
          acc = fma(r, r, acc);
        }
        const double err = sqrt(acc * 0.25);
        const bool finite = finite4(yn[0], yn[1], yn[2], yn[3]) && finite4(dy[0], dy[1], dy[2], dy[3]) && isfinite(err);
        const bool accept = forced ? finite : (finite && err <= 1.0);
        if (forced && !finite) {
          st = GC_ST_NONFINITE_;
        } else if (accept) {
          const double sc = scale_after_accept(err);
          const double h_next = prev_rejected ? h_try * fmin(sc, 1.0) : h_try * sc;
          if (p.poincare_capacity > 0 && p.section == 1) {              // O8b: bounce section
            if (bounce_crossed(y[3], yn[3])) {
              double hk1[4], hk7[4], hd[4];
#pragma unroll
              for (int c = 0; c < 4; ++c) {
                hk1[c] = h_try * GC_K(0, c); hk7[c] = h_try * GC_K(6, c); hd[c] = dense_hd(kbuf, c, h_try);
              }
              bounce_emit(y, yn, hk1, hk7, hd, i, t, h_try, p.poincare, p.poincare_capacity, p.poincare_count);
            }
          } else if (p.poincare_capacity > 0 && floor(y[2] / 6.283185307179586476925286766559) !=
                                                    floor(yn[2] / 6.283185307179586476925286766559)) {
            Dense3 d;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
              d.r1[c] = y[c];
              d.r2[c] = yn[c] - y[c];
              d.r3[c] = h_try * GC_K(0, c) - d.r2[c];
              d.r4[c] = d.r2[c] - h_try * GC_K(6, c) - d.r3[c];
              d.r5[c] = dense_hd(kbuf, c, h_try);
            }
            poincare_emit(d, i, t, h_try, y[2], yn[2], p.poincare, p.poincare_capacity, p.poincare_count);
          }
          const double t_new = clipped ? p.t_max : t + h_try;
          if (p.nsamp > 0 && jn < p.nsamp && sample_time(p, jn) <= t_new) {       // O9
            double hd[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) hd[c] = dense_hd(kbuf, c, h_try);
            while (jn < p.nsamp) {
              const double tj = sample_time(p, jn);
              if (tj > t_new) break;
              const double tau = (tj - t) / h_try;
#pragma unroll
              for (int c = 0; c < 4; ++c) {
                const double v = dense_component(y[c], yn[c], h_try * GC_K(0, c), h_try * GC_K(6, c), hd[c], tau);
                p.samples[((long long)c * p.nsamp + jn) * p.n + i] = c == 3 ? v * p.v_ref : v;
              }
              ++jn;
            }
          }
          const bool lost_now = yn[0] >= p.s_loss;
          double t_rep = t_new;
          if (lost_now && p.refine_loss && y[0] < p.s_loss) {            // O7b
            double hd[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) hd[c] = dense_hd(kbuf, c, h_try);
            const double tau = loss_root(y[0], yn[0], h_try * GC_K(0, 0), h_try * GC_K(6, 0), hd[0], p.s_loss);
#pragma unroll
            for (int c = 0; c < 4; ++c)
              yn[c] = dense_component(y[c], yn[c], h_try * GC_K(0, c), h_try * GC_K(6, c), hd[c], tau);
            t_rep = fma(tau, h_try, t);
          }
          t = lost_now ? t_rep : t_new;
#pragma unroll
          for (int c = 0; c < 4; ++c) { y[c] = yn[c]; GC_K(0, c) = GC_K(6, c); }      // FSAL
          ++n_acc;
          if (forced) ++n_forced;
          prev_rejected = false;
          if (!clipped) h = h_next;
          if (h < p.h_min) h = p.h_min;
          if (lost_now) st = 1;
          else if (y[0] <= p.s_min) st = 2;
          else if (clipped) st = 0;
          else if (attempts >= p.max_steps) st = 3;
        } else {
          ++n_rej;
          h = h_try * scale_after_reject(err);
          if (h < p.h_min) h = p.h_min;
          prev_rejected = true;
          if (attempts >= p.max_steps) st = 3;
        }
      }
    }

    // ---- a particle that stopped: store its results, free the lane ------------------------------------------------
    if (i >= 0 && st >= 0) {
      p.y_out[0 * p.n + i] = y[0];
      p.y_out[1 * p.n + i] = y[1];
      p.y_out[2 * p.n + i] = y[2];
      p.y_out[3 * p.n + i] = y[3] * p.v_ref;
      p.t_out[i] = t;
      p.status[i] = st;
      if (p.h_inout) p.h_inout[i] = h;
      if (p.n_acc) p.n_acc[i] = (p.resume ? p.n_acc[i] : 0) + n_acc;
      if (p.n_rej) p.n_rej[i] = (p.resume ? p.n_rej[i] : 0) + n_rej;
      if (p.n_forced) p.n_forced[i] = (p.resume ? p.n_forced[i] : 0) + n_forced;
      if (p.nsamp > 0 && p.sample_end) p.sample_end[i] = (int)jn;
      i = -1;
    }
  }
}

#undef GC_K

}  // namespace gc
