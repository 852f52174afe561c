// field.cuh -- device-side view of a gc_field and the launch parameter blocks.
#pragma once
#include <stdint.h>

namespace gc {

// Device pointers into the tables owned by gc_field.  Passed to kernels by value.
struct FieldDev {
  int ns, nfp, nh, nk;
  double psi0, inv_psi0;
  // as given by the caller (generic kernel, gc_field_eval)
  const int* xm;         // [nh]
  const int* xn;         // [nh]
  const double* bmnc;    // [ns][nh]
  const double* G;       // [ns]
  const double* I;       // [ns]
  const double* iota;    // [ns]
  const int* mode_m;     // [nk]
  const int* mode_n;     // [nk]
  const double* omega;   // [nk]
  const double* inv_omega;  // [nk] 1 / omega (mma kernel: no division per mode and right-hand side)
  const double* phase;   // [nk]
  const double* phihat;  // [ns][nk]
  // NEXT-4: sin coefficients of B and the covariant radial component K (nullptr = absent), [ns][nh] each
  const double* bmns;
  const double* kmnc;
  const double* kmns;
  // the same four tables with the row stride padded to nhp = roundup4(nh) (zero fill) and 32-byte aligned rows, so the
  // lane kernel and the point evaluations read FOUR consecutive harmonics of a node row with one 256-bit load
  // (nullptr = absent); xmp / xnp are xm / xn padded with (0, 0) harmonics
  const double* bmnc4;
  const double* bmns4;
  const double* kmnc4;
  const double* kmns4;
  const int* xmp;
  const int* xnp;
  int nhp;
  // packed by-node layout of the warp kernel (kernels_warp.cuh): rows[node][it][lane]
  const double* rows;
  int M, N;              // max xm, max |xn|
  int cl_log;            // log2(lanes per m-group)
  int nit_main, nx, nit; // main iterations, extra iterations, total
  // per-cell window images of the tile kernel (kernels_tile.cuh): images[cell][10 E] doubles,
  // [E][6] rows cell-1..cell+4 then [E][4] rows cell..cell+3; entry e = m (1 + 2 NMAX) + {0 | 2n-1 | 2n},
  // then G, I, iota, then the nk mode amplitudes
  const double* tile_images;
  int tile_E, tile_nmax;
  // by-node image of the mma kernel (kernels_mma.cuh): image[ns + 4][mma_RS], image row = node + 2 (two zero rows
  // at either end); a row holds the DMMA B fragments (P, Q)(m >= 1, n >= 1), b(m, 0), b(0, n), G, I, iota, modes
  const double* mma_image;
  int mma_RS, mma_MT, mma_KS;
  // NEXT-4: images of the same row layout (fragments, b(m, 0), b(0, n) only) for bmns, kmnc, kmns; nullptr = absent
  const double* mma_image_bs;
  const double* mma_image_kc;
  const double* mma_image_ks;
  // NEXT-2 (kernels_grid.cuh): node values of B on the (s, theta, zeta) grid over one field period in the gather
  // layout grid[ngs][nth + 3][nze][4] (entry k = nodes k .. k+3 mod nze; three theta rows repeated); nullptr = the
  // direct harmonic sum.  th_scale = nth / 2 pi, ze_scale = nze nfp / 2 pi (nodes per radian).
  // grid_kind 1: the Lagrange gather layout above.  grid_kind 2 (reading A31, C1 tricubic Hermite): grid[ngs][nth + 1]
  // [nze + 1][8], per node (f, f_ze, f_th, f_th_ze, f_s, f_s_ze, f_s_th, f_s_th_ze) pre-multiplied by the cell widths of
  // the differentiated directions (64 bytes = two 256-bit loads), one periodic image appended in both angles.
  const double* grid;
  int grid_kind;
  double inv_ds, inv_dth, inv_dze;   // 1 / cell width in s, theta, zeta (Hermite: derivative outputs)
  int ngs, nth, nze;
  double th_scale, ze_scale, inv_nth, inv_nze;
};

// Integrator parameters as the kernels see them (gc_trace_params + derived values).
struct TraceDev {
  double mass, charge, t0, t_max, rtol, atol, v_ref, inv_v_ref, h0, h_min, s_loss, s_min;
  long long max_steps, poincare_capacity;
  long long n;
  int resume;                         // GC_TRACE_RESUME: skip particles whose status is not 0 on entry
  int section;                        // Poincare records: 0 zeta = 0 mod 2 pi (O8), 1 v_par = 0 (O8b)
  int refine_loss;                    // O7b: lost particles report the root of s(tau) = s_loss of their last step
  const double *s0, *th0, *ze0, *vpar0, *mu;
  double* h_inout;
  double *y_out, *t_out;
  int* status;
  int *n_acc, *n_rej, *n_forced;
  double* poincare;
  unsigned long long* poincare_count;
  unsigned long long* work_counter;   // persistent-kernel particle queue head
  // O9 (gc_trace_sampled): samples[4][nsamp][n] at tau_j = fma(j, sample_dt, sample_t0); nsamp = 0 disables
  double sample_t0, sample_dt;
  long long nsamp;
  double* samples;
  int* sample_end;
  // the symplectic integrator inside the cell-binned body (trace_mma_symplectic_kernel): fixed step, steps per call,
  // tolerance and cap of the quasi-Newton iteration, chi at the radial nodes; n_acc / n_rej receive steps / iterations
  double sym_dt, sym_tol;
  long long sym_nsteps;
  int sym_max_iter;
  const double* chi;
};

}  // namespace gc
