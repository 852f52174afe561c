// kernels_grid.cuh -- NEXT-2 of SURVEY.md section 8(f): B as a local tricubic interpolant of its own node values
// ("CUDA kernels implement field interpolation and trajectory integration on GPU" PAPER.md:48; "local tricubics"
// PAPER.md:80,111; reading A27 of DESIGN.md).
//
// Grid: s_i = i / (ngs - 1), theta_j = 2 pi j / nth, zeta_k = (2 pi / nfp) k / nze, one field period, both angles
// periodic.  Node values are the direct harmonic sum O2 (grid_build_kernel).  Evaluation is the tensor product of
// the cubic Lagrange weights of O1 in each direction: the radial stencil is clamped as in O1, an angular stencil is
// the four nodes c-1 .. c+2 around the cell c = floor(angle * nodes_per_radian), taken modulo the period.
//
// Layout in HBM / L2: grid[ngs][nth + 3][nze][4] doubles: entry (i, j, k) holds the FOUR consecutive zeta nodes
// k .. k+3 (mod nze) of row (i, j mod nth), 32-byte aligned, and the first three theta rows are repeated at the end.
// A stencil is then 16 aligned 32-byte runs, each fetched by ONE 256-bit load (LDG.E.256, sm_100): 16 load
// instructions per evaluation instead of 64, no modulo in the hot loop, every load exactly one sector.  The table is
// four times the node count (54 MB for 101 x 128 x 128) and lives in the 126 MB L2.  This path is gather-bound (64
// doubles per right-hand side through the L1 data pipe), not FP64-bound like the harmonic sum: 192 FMA per
// evaluation of B and its three derivatives.
#pragma once
#include "device_math.cuh"
#include "field.cuh"

namespace gc {

// Cubic Lagrange weights on a periodic uniform grid: first node j0 in [0, nodes), weights w[4] and d/d(angle)
// weights dw[4]; x = u - (c - 1) lies in [1, 2), so the stencil is always centred.  The decision floor(u) is taken
// on the same single product angle * npr as in the oracle.
__device__ __forceinline__ void periodic_weights(int nodes, double inv_nodes, double npr, double angle, int& j0,
                                                 double w[4], double dw[4]) {
  const double u = angle * npr;
  const double c1 = floor(u) - 1.0;
  const double x = u - c1, x1 = x - 1.0, x2 = x - 2.0, x3 = x - 3.0;
  w[0] = -(x1 * x2 * x3) * (1.0 / 6.0);
  w[1] = (x * x2 * x3) * 0.5;
  w[2] = -(x * x1 * x3) * 0.5;
  w[3] = (x * x1 * x2) * (1.0 / 6.0);
  dw[0] = -(x2 * x3 + x1 * x3 + x1 * x2) * (npr / 6.0);
  dw[1] = (x2 * x3 + x * x3 + x * x2) * (npr * 0.5);
  dw[2] = -(x1 * x3 + x * x3 + x * x1) * (npr * 0.5);
  dw[3] = (x1 * x2 + x * x2 + x * x1) * (npr / 6.0);
  // (c - 1) mod nodes without an integer division: both are integers below 2^53, so the fma is exact and the
  // quotient estimate is off by at most one
  const double nd = (double)nodes;
  double r = fma(-floor(c1 * inv_nodes), nd, c1);
  if (r < 0.0) r += nd;
  if (r >= nd) r -= nd;
  j0 = (r >= 0.0 && r < nd) ? (int)r : 0;          // NaN / inf angles: any valid row (the weights are NaN anyway)
}

// Four consecutive doubles from a 32-byte aligned address of read-only memory in one instruction.
__device__ __forceinline__ void ldg256(const double* p, double& a, double& b, double& c, double& d) {
  asm("ld.global.nc.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}

// out = B, dB/ds, dB/dtheta, dB/dzeta from the 64 nodes around (s, theta, zeta).
__device__ __forceinline__ void eval_B_grid(const FieldDev& f, double s, double th, double ze, double out[4]) {
  int i0, j0, k0;
  double ws[4], dws[4], wt[4], dwt[4], wz[4], dwz[4];
  lagrange_weights(f.ngs, s, i0, ws, dws);
  periodic_weights(f.nth, f.inv_nth, f.th_scale, th, j0, wt, dwt);
  periodic_weights(f.nze, f.inv_nze, f.ze_scale, ze, k0, wz, dwz);
  const size_t rs = (size_t)f.nze * 4, ps = (size_t)(f.nth + 3) * rs;
  const double* base = f.grid + (size_t)i0 * ps + (size_t)j0 * rs + (size_t)k0 * 4;
  double B = 0.0, Bs = 0.0, Bt = 0.0, Bz = 0.0;
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    double ra = 0.0, rat = 0.0, raz = 0.0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      double v0, v1, v2, v3;
      ldg256(base + a * ps + b * rs, v0, v1, v2, v3);
      const double v = fma(wz[3], v3, fma(wz[2], v2, fma(wz[1], v1, wz[0] * v0)));
      const double vz = fma(dwz[3], v3, fma(dwz[2], v2, fma(dwz[1], v1, dwz[0] * v0)));
      ra = fma(wt[b], v, ra);
      rat = fma(dwt[b], v, rat);
      raz = fma(wt[b], vz, raz);
    }
    B = fma(ws[a], ra, B);
    Bs = fma(dws[a], ra, Bs);
    Bt = fma(ws[a], rat, Bt);
    Bz = fma(ws[a], raz, Bz);
  }
  out[0] = B; out[1] = Bs; out[2] = Bt; out[3] = Bz;
}

// ---- reading A31: the C1 tricubic Hermite interpolant --------------------------------------------------------------
// 1-D cubic Hermite basis on [0, 1] and its derivative: h[corner][order] (value / slope at corner 0 / 1).
__device__ __forceinline__ void hermite_basis(double x, double (&h)[2][2], double (&dh)[2][2]) {
  const double x2 = x * x, x3 = x2 * x;
  h[0][0] = fma(2.0, x3, fma(-3.0, x2, 1.0));  dh[0][0] = 6.0 * (x2 - x);
  h[1][0] = fma(-2.0, x3, 3.0 * x2);           dh[1][0] = 6.0 * (x - x2);
  h[0][1] = x3 - 2.0 * x2 + x;                 dh[0][1] = fma(3.0, x2, fma(-4.0, x, 1.0));
  h[1][1] = x3 - x2;                           dh[1][1] = fma(3.0, x2, -2.0 * x);
}

// cell index in [0, nodes) and local coordinate of a periodic direction; the decision floor(u) on the same product as
// the oracle
__device__ __forceinline__ void periodic_cell(int nodes, double inv_nodes, double npr, double angle, int& c, double& x) {
  const double u = angle * npr, fl = floor(u);
  x = u - fl;
  const double nd = (double)nodes;
  double r = fma(-floor(fl * inv_nodes), nd, fl);
  if (r < 0.0) r += nd;
  if (r >= nd) r -= nd;
  c = (r >= 0.0 && r < nd) ? (int)r : 0;
}

// out = B, dB/ds, dB/dtheta, dB/dzeta from the 8 corner nodes (64 doubles, 16 x 256-bit loads) of the cell.
__device__ __forceinline__ void eval_B_hermite(const FieldDev& f, double s, double th, double ze, double out[4]) {
  const double us = s * (double)(f.ngs - 1);
  double cs = floor(us);
  if (!(cs >= 0.0)) cs = 0.0;                                  // also NaN
  if (cs > (double)(f.ngs - 2)) cs = (double)(f.ngs - 2);
  const int ci = (int)cs;
  const double x = us - cs;
  int cj, ck;
  double y, z;
  periodic_cell(f.nth, f.inv_nth, f.th_scale, th, cj, y);
  periodic_cell(f.nze, f.inv_nze, f.ze_scale, ze, ck, z);
  double hs[2][2], dhs[2][2], ht[2][2], dht[2][2], hz[2][2], dhz[2][2];
  hermite_basis(x, hs, dhs);
  hermite_basis(y, ht, dht);
  hermite_basis(z, hz, dhz);
  const size_t rs = (size_t)(f.nze + 1) * 8, ps = (size_t)(f.nth + 1) * rs;
  const double* base = f.grid + (size_t)ci * ps + (size_t)cj * rs + (size_t)ck * 8;
  double B = 0.0, Bs = 0.0, Bt = 0.0, Bz = 0.0;
#pragma unroll
  for (int a = 0; a < 2; ++a) {
    double w[2] = {0.0, 0.0}, wt[2] = {0.0, 0.0}, wz[2] = {0.0, 0.0};      // by s-order p
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      const double* nd0 = base + a * ps + b * rs;                           // node (a, b, 0); (a, b, 1) follows it
#pragma unroll
      for (int p = 0; p < 2; ++p) {
        double d0[4], d1[4];                                                // (q, r) = (0,0) (0,1) (1,0) (1,1)
        ldg256(nd0 + 4 * p, d0[0], d0[1], d0[2], d0[3]);
        ldg256(nd0 + 8 + 4 * p, d1[0], d1[1], d1[2], d1[3]);
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          const double v = fma(hz[1][1], d1[2 * q + 1], fma(hz[1][0], d1[2 * q], fma(hz[0][1], d0[2 * q + 1],
                               hz[0][0] * d0[2 * q])));
          const double vz = fma(dhz[1][1], d1[2 * q + 1], fma(dhz[1][0], d1[2 * q], fma(dhz[0][1], d0[2 * q + 1],
                                dhz[0][0] * d0[2 * q])));
          w[p] = fma(ht[b][q], v, w[p]);
          wt[p] = fma(dht[b][q], v, wt[p]);
          wz[p] = fma(ht[b][q], vz, wz[p]);
        }
      }
    }
#pragma unroll
    for (int p = 0; p < 2; ++p) {
      B = fma(hs[a][p], w[p], B);
      Bs = fma(dhs[a][p], w[p], Bs);
      Bt = fma(hs[a][p], wt[p], Bt);
      Bz = fma(hs[a][p], wz[p], Bz);
    }
  }
  out[0] = B; out[1] = Bs * f.inv_ds; out[2] = Bt * f.inv_dth; out[3] = Bz * f.inv_dze;
}

// B from whichever interpolant the field carries (grid_kind 1 or 2).
template <int KIND>
__device__ __forceinline__ void eval_B_interp(const FieldDev& f, double s, double th, double ze, double out[4]) {
  if (KIND == 2) eval_B_hermite(f, s, th, ze, out);
  else eval_B_grid(f, s, th, ze, out);
}
__device__ __forceinline__ void eval_B_interp_rt(const FieldDev& f, double s, double th, double ze, double out[4]) {
  if (f.grid_kind == 2) eval_B_hermite(f, s, th, ze, out);
  else eval_B_grid(f, s, th, ze, out);
}

}  // namespace gc
