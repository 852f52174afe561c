// kernels_mma.cuh -- hot-path kernel for large ensembles, second generation: the harmonic sum as FP64 matrix
// instructions (DMMA.8x8x4), eight particles per instruction.
//
// Why.  kernels_tile.cuh is bound by shared-memory operand delivery: every DFMA of its sweep takes one operand
// that each lane loads for itself (2 DFMA per loaded double; profiles/r1_ncu_tile_config1.md).  Once particles
// are binned by radial cell the inner sum IS a small dense contraction: with
//     b(m,n) cos(m th - n ph) + b(m,-n) cos(m th + n ph) = P c_m C_n + Q s_m S_n          (ph = nfp zeta)
// and radial interpolation commuting with the harmonic sum, for every node row r of the stencil and poloidal
// number m the sweep needs
//     PC[p][r,m] = sum_n C_n(p) P[r][m,n]     PS = sum_n n S_n(p) P     QS = sum_n S_n(p) Q     QC = sum_n n C_n(p) Q
// i.e. D[8 particles][8 columns (r, m)] += A[8 particles][4 toroidal numbers] * B[4 toroidal numbers][8 columns]:
// mma.sync.m8n8k4.f64.  The A operand is per-particle trigonometry held in registers, the B operand is the
// table, identical for the eight particles of a group and fetched ONCE per group (one 16-byte load per lane feeds
// four DMMA = 32 DFMA-equivalents per lane), the accumulators never leave registers.  On B200 DMMA.8x8x4 shares
// the FP64 units with DFMA (37 TFLOP/s measured for either, 35 when mixed: same roofline), so this buys operand
// bandwidth, not peak; latency 26 cycles, two independent accumulators saturate the pipe (measured).
//
// Layout of the work.  As in kernels_tile.cuh a lane owns a particle for everything that is per particle
// (Lagrange weights, one sincos(theta) and one sincos(nfp zeta), profiles, perturbation, guiding-centre algebra,
// Dormand-Prince controller).  Only the harmonic sum changes hands: a warp pushes its 32 particles through the
// sweep in four GROUPS of eight.  For group G lane = 4 g + q plays the FRAGMENT role for particle 8 G + g:
//   * it fetches that particle's (cos, sin)(theta), (cos, sin)(nfp zeta) by shuffle and builds, by complex
//     powers, the A operands C_n, S_n, n C_n, n S_n for n = 4 j + q + 1 (k-step j) and (c_m, s_m) for its four
//     poloidal numbers m = 1 + 8 T + 2 q + e;
//   * DMMA fragments: A[g][q], B[q][g], D[g][2q, 2q+1]; the B fragments (P, Q)(m, n) sit in the image in lane
//     order, one 16-byte load per lane and k-step; n = 0 initialises the PC accumulator, m = 0 is a 16-term DFMA
//     sum split over the quad;
//   * rows: the group sweeps the UNION of the stencil rows of its 8 particles (4 rows when they share a stencil,
//     5 when they straddle a node); the Lagrange weights of a row come from the particle's six-entry table in
//     shared memory (one LDS.128) and are exactly 0 for a row outside that particle's stencil, so a particle's
//     result does not depend on who it shares a group with;
//   * per row the epilogue turns the eight accumulators of a lane into its share of B, B_s, B_theta, B_zeta;
//     two butterfly shuffles sum the quad and one more hands the four sums back to the particle lane.
// Window: the 8 node rows cell-2 .. cell+5 of a by-node image (contiguous in global memory, ONE bulk TMA copy per
// cell change); stencils that start further than 2 rows from the tile's cell are swept from global memory with the
// same instruction sequence (bit-identical results).  Binning, epochs, tiles, records and the integrator are
// trace_binned_body of kernels_tile.cuh; tiles are 64 particles (two warps share a window; fewer when the ensemble
// cannot fill the grid), chunks are 8 attempts: frequent re-binning keeps the groups on 4-row unions and parks few
// particles.
#pragma once
#include <cooperative_groups.h>

#include <type_traits>

#include "device_math.cuh"
#include "field.cuh"
#include "kernels_generic.cuh"
#include "kernels_tile.cuh"      // TileScratch, record layout, mbarrier / bulk-copy helpers, home_bin, cDp*

namespace gc {

#ifndef GC_MMA_THREADS
#define GC_MMA_THREADS 64
#endif
#ifndef GC_MMA_MINB
#define GC_MMA_MINB 4
#endif
constexpr int kMmaThreads = GC_MMA_THREADS;      // particles per tile = threads per block (2 warps share a window)
constexpr int kMmaBlocksPerSm = GC_MMA_MINB;     // 8 warps per SM at <= 255 registers
#ifndef GC_MMA_CAP
#define GC_MMA_CAP 8
#endif
constexpr int kMmaCap = GC_MMA_CAP;              // attempted steps per particle per chunk (short: re-binning keeps the
                                                 // groups on 4-row unions and parks fewer particles)
constexpr int kMmaWinRows = 8;                   // node rows cell-2 .. cell+5
constexpr int kMmaWtab = 6;                      // (w, dw) entries of a particle's weight table in shared memory
constexpr int kMmaNone = 1 << 20;                // "no stencil": a row offset that gives weight 0 on every row

// Offsets (in doubles) inside one node row of the image; RS = row stride.
template <int MT, int KS>
struct MmaRow {
  static constexpr int kFrag = 0;                      // [MT][KS][32 lanes][2]: (P, Q)(m = 1 + 8T + lane/4, n = 4j + lane%4 + 1)
  static constexpr int kN0 = MT * KS * 64;             // [8 MT]: b(m, 0), m = 1 .. 8 MT
  static constexpr int kM0 = kN0 + 8 * MT;             // [4 KS + 1]: b(0, n), n = 0 .. 4 KS
  static constexpr int kProf = kM0 + 4 * KS + 1;       // G, I, iota
  static constexpr int kModes = kProf + 3;             // [nk]
  static __host__ __device__ int stride(int nk) { return (kModes + nk + 1) & ~1; }
};

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

struct LdS {
  static __device__ __forceinline__ double2 ld2(const double* p) { return *reinterpret_cast<const double2*>(p); }
  static __device__ __forceinline__ double ld1(const double* p) { return *p; }
};
struct LdG {
  static __device__ __forceinline__ double2 ld2(const double* p) { return __ldg(reinterpret_cast<const double2*>(p)); }
  static __device__ __forceinline__ double ld1(const double* p) { return __ldg(p); }
};

__device__ __forceinline__ double quad_sum(double v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  return v;
}
// (a + i b)(c + i d)
__device__ __forceinline__ void cmul(double a, double b, double c, double d, double& re, double& im) {
  re = fma(a, c, -b * d);
  im = fma(a, d, b * c);
}


// One pass over node rows r_lo .. r_hi (warp-uniform) of the image at `base` (row r at base + r RS) for the group of
// 8 particles whose lanes are 8 G .. 8 G + 7, executed by the lanes in their FRAGMENT role (g = lane / 4,
// q = lane % 4, serving particle 8 G + g).  wsrc = that particle's weight table in shared memory (6 x (w, dw):
// zero, the four stencil weights, zero), off_f = row of its first stencil node in this pass (kMmaNone when it does
// not take part: weight 0 on every row).  Issues the DMMA and accumulates this lane's share of B, B_s, B_theta,
// B_zeta / nfp in o[].
// SIN (NEXT-4): the image holds the coefficients of a sin series, b sin(m th - n ph): the caller passes (c_m, s_m)
// rotated by a quarter period, (s_m, -c_m), which turns the cos sweep into the sin sweep for every m >= 1; only the
// m = 0 row differs: b(0, n) sin(-n ph) = -b S_n, zeta-derivative -n nfp b C_n.
template <int MT, int KS, class Ld, bool SIN = false>
__device__ __forceinline__ void mma_sweep(const double* base, int RS, int r_lo, int r_hi, int off_f,
                                          const double2* wsrc, int lane, int q,
                                          const double (&AC)[KS], const double (&AS)[KS], const double (&AnC)[KS],
                                          const double (&AnS)[KS], const double (&cm)[2 * MT],
                                          const double (&sm)[2 * MT], double (&o)[4]) {
  using R = MmaRow<MT, KS>;
  double mc[2 * MT], ms[2 * MT];                       // m c_m, m s_m of this lane's columns m = 1 + 8 T + 2 q + e
#pragma unroll
  for (int k = 0; k < 2 * MT; ++k) {
    const double m = (double)(1 + 8 * (k >> 1) + 2 * q + (k & 1));
    mc[k] = m * cm[k];
    ms[k] = m * sm[k];
  }
#ifndef GC_MMA_ROW_UNROLL
#define GC_MMA_ROW_UNROLL 2
#endif
  constexpr int kRowUnroll = GC_MMA_ROW_UNROLL;
#pragma unroll kRowUnroll
  for (int r = r_lo; r <= r_hi; ++r) {
    // (w, dw) of row r for the particle this lane serves: entries 1..4 of its table are the stencil weights,
    // entries 0 and 5 are zero (rows outside the stencil)
    const double2 wd = wsrc[min(max(r - off_f, -1), 4) + 1];
    const double wr = wd.x, dwr = wd.y;
    const double* row = base + (size_t)r * RS;
    double T1 = 0.0, T2 = 0.0, T3 = 0.0;
#pragma unroll
    for (int T = 0; T < MT; ++T) {
      const double2 ini = Ld::ld2(row + R::kN0 + 8 * T + 2 * q);
      double PC0 = ini.x, PC1 = ini.y, PS0 = 0.0, PS1 = 0.0, QS0 = 0.0, QS1 = 0.0, QC0 = 0.0, QC1 = 0.0;
#pragma unroll
      for (int j = 0; j < KS; ++j) {
        const double2 pq = Ld::ld2(row + R::kFrag + ((T * KS + j) * 32 + lane) * 2);
        dmma884(PC0, PC1, AC[j], pq.x);
        dmma884(PS0, PS1, AnS[j], pq.x);
        dmma884(QS0, QS1, AS[j], pq.y);
        dmma884(QC0, QC1, AnC[j], pq.y);
      }
      // columns m = 1 + 8 T + 2 q + e  (index 2 T + e of cm / sm)
      const double c0 = cm[2 * T], s0 = sm[2 * T], c1 = cm[2 * T + 1], s1 = sm[2 * T + 1];
      T1 = fma(c0, PC0, T1); T1 = fma(s0, QS0, T1);
      T1 = fma(c1, PC1, T1); T1 = fma(s1, QS1, T1);
      T2 = fma(mc[2 * T], QS0, T2); T2 = fma(-ms[2 * T], PC0, T2);
      T2 = fma(mc[2 * T + 1], QS1, T2); T2 = fma(-ms[2 * T + 1], PC1, T2);
      T3 = fma(s0, QC0, T3); T3 = fma(-c0, PS0, T3);
      T3 = fma(s1, QC1, T3); T3 = fma(-c1, PS1, T3);
    }
    // m = 0: b(0,n) C_n and its zeta-derivative, n = 4 j + q + 1 on this lane; n = 0 on lane q = 0
    double x = (!SIN && q == 0) ? Ld::ld1(row + R::kM0) : 0.0, xs = 0.0;
#pragma unroll
    for (int j = 0; j < KS; ++j) {
      const double b0 = Ld::ld1(row + R::kM0 + 1 + 4 * j + q);
      if constexpr (SIN) {
        x = fma(-b0, AS[j], x);
        xs = fma(b0, AnC[j], xs);
      } else {
        x = fma(b0, AC[j], x);
        xs = fma(b0, AnS[j], xs);
      }
    }
    T1 += x;
    T3 -= xs;
    o[0] = fma(wr, T1, o[0]);
    o[1] = fma(dwr, T1, o[1]);
    o[2] = fma(wr, T2, o[2]);
    o[3] = fma(wr, T3, o[3]);
  }
}

// Right-hand side of one lane = one particle (same contract as rhs_tile); must be called by all 32 lanes of a warp.
// win = shared-memory copy of image rows cell .. cell+7 (node rows cell-2 .. cell+5).
// FIELD_ONLY (the symplectic integrator, NEXT-3): stop after the sums and the profiles and hand out B, B_s, B_theta,
// B_zeta in dy[0..3] and G, G_s, I, I_s, iota, iota_s in *prof_out instead of the guiding-centre algebra.
template <int MT, int KS, bool MODES, bool EXTRA = false, bool FIELD_ONLY = false>
__device__ __forceinline__ void rhs_mma(const FieldDev& f, const double* win, double* ext, int cell, bool active,
                                        double mass, double charge, double mu, double v_ref, double inv_v_ref,
                                        double t, const double (&y)[4], double (&dy)[4], Profiles* prof_out = nullptr) {
  using R = MmaRow<MT, KS>;
  const int lane = threadIdx.x & 31, q = lane & 3;
  const int RS = f.mma_RS;
  // ---- particle role: stencil, weights, one sincos(theta), one sincos(nfp zeta) ------------------------------------
  int i0;
  double w[4], dw[4];
  lagrange_weights(f.ns, active ? y[0] : 0.0, i0, w, dw);
  const int off = i0 - cell + 2;
  const bool inwin = active && off >= 0 && off <= kMmaWinRows - 4;
  const bool outside = active && !inwin;
  // weight table of this particle for the fragment lanes: [0] = [5] = 0, [1 + a] = (w[a], dw[a])
  double2* wtab = reinterpret_cast<double2*>(ext) + (size_t)threadIdx.x * kMmaWtab;
  __syncwarp();                                                         // fragment lanes are done with the last table
  wtab[0] = make_double2(0.0, 0.0);
#pragma unroll
  for (int a = 0; a < 4; ++a) wtab[1 + a] = make_double2(w[a], dw[a]);
  wtab[5] = make_double2(0.0, 0.0);
  __syncwarp();
  const double thr = active ? reduce_2pi(y[1]) : 0.0;                 // idle lanes offer finite operands
  const double phr = active ? reduce_2pi((double)f.nfp * y[2]) : 0.0;
  double c1, s1, C1, S1;
  sincos_poly(thr, s1, c1);
  sincos_poly(phr, S1, C1);
  double fb[4] = {0.0, 0.0, 0.0, 0.0};
  double fk[4] = {0.0, 0.0, 0.0, 0.0};                                  // EXTRA: the K series
  const unsigned onmask = __ballot_sync(0xffffffffu, active);
#pragma unroll 1
  for (int G = 0; G < 4; ++G) {
    if (((onmask >> (8 * G)) & 0xFFu) == 0u) continue;                // warp-uniform
    const int src = 8 * G + (lane >> 2);
    const bool ingrp = (lane >> 3) == G;
    const double2* wsrc = wtab + ((src - lane) * kMmaWtab);           // table of particle src (same warp)
    // ---- fragment role: trigonometry of particle src for n = 4 j + q + 1 and m = 1 + 8 T + 2 q + e -----------------
    const double gc1 = __shfl_sync(0xffffffffu, c1, src), gs1 = __shfl_sync(0xffffffffu, s1, src);
    const double gC1 = __shfl_sync(0xffffffffu, C1, src), gS1 = __shfl_sync(0xffffffffu, S1, src);
    double AC[KS], AS[KS], AnC[KS], AnS[KS], cm[2 * MT], sm[2 * MT];
    {
      double e2r, e2i, e3r, e3i, e4r, e4i;
      cmul(gC1, gS1, gC1, gS1, e2r, e2i);
      cmul(e2r, e2i, gC1, gS1, e3r, e3i);
      cmul(e2r, e2i, e2r, e2i, e4r, e4i);
      AC[0] = q == 0 ? gC1 : q == 1 ? e2r : q == 2 ? e3r : e4r;
      AS[0] = q == 0 ? gS1 : q == 1 ? e2i : q == 2 ? e3i : e4i;
#pragma unroll
      for (int j = 1; j < KS; ++j) cmul(AC[j - 1], AS[j - 1], e4r, e4i, AC[j], AS[j]);
#pragma unroll
      for (int j = 0; j < KS; ++j) {
        const double n = (double)(4 * j + q + 1);
        AnC[j] = n * AC[j];
        AnS[j] = n * AS[j];
      }
      double f2r, f2i, f3r, f3i, f5r, f5i, f7r, f7i;
      cmul(gc1, gs1, gc1, gs1, f2r, f2i);
      cmul(f2r, f2i, gc1, gs1, f3r, f3i);
      cmul(f3r, f3i, f2r, f2i, f5r, f5i);
      cmul(f5r, f5i, f2r, f2i, f7r, f7i);
      cm[0] = q == 0 ? gc1 : q == 1 ? f3r : q == 2 ? f5r : f7r;
      sm[0] = q == 0 ? gs1 : q == 1 ? f3i : q == 2 ? f5i : f7i;
      cmul(cm[0], sm[0], gc1, gs1, cm[1], sm[1]);
      if constexpr (MT == 2) {
        double f4r, f4i, f8r, f8i;
        cmul(f2r, f2i, f2r, f2i, f4r, f4i);
        cmul(f4r, f4i, f4r, f4i, f8r, f8i);
        cmul(cm[0], sm[0], f8r, f8i, cm[2], sm[2]);
        cmul(cm[1], sm[1], f8r, f8i, cm[3], sm[3]);
      }
    }
    double o[4] = {0.0, 0.0, 0.0, 0.0};
    // ---- in-window stencils of the group: one sweep over the union of their rows ---------------------------------
    const int r_lo = __reduce_min_sync(0xffffffffu, (ingrp && inwin) ? off : kMmaNone);
    const int r_hi = __reduce_max_sync(0xffffffffu, (ingrp && inwin) ? off + 3 : -1);
    if (r_hi >= 0) {
      const int off_f = __shfl_sync(0xffffffffu, inwin ? off : kMmaNone, src);
      mma_sweep<MT, KS, LdS>(win, RS, r_lo, r_hi, off_f, wsrc, lane, q, AC, AS, AnC, AnS, cm, sm, o);
    }
    // ---- stencils outside the window: one sweep per distinct stencil, rows from global memory ----------------------
    unsigned pend = __ballot_sync(0xffffffffu, ingrp && outside);
    while (pend) {
      const int i0L = __shfl_sync(0xffffffffu, i0, __ffs(pend) - 1);
      const bool mine = ingrp && outside && i0 == i0L;
      const int off_f = __shfl_sync(0xffffffffu, mine ? 0 : kMmaNone, src);
      mma_sweep<MT, KS, LdG>(f.mma_image + (size_t)(i0L + 2) * RS, RS, 0, 3, off_f, wsrc, lane, q, AC, AS, AnC, AnS,
                             cm, sm, o);
      pend &= ~__ballot_sync(0xffffffffu, mine);
    }
    // ---- NEXT-4: the sin series of B and the two series of K, same rows, images read through L1 -------------------
    double ok[4] = {0.0, 0.0, 0.0, 0.0};
    if constexpr (EXTRA) {
      const int off_w = __shfl_sync(0xffffffffu, inwin ? off : kMmaNone, src);
      const unsigned pend0 = __ballot_sync(0xffffffffu, ingrp && outside);
      double cr[2 * MT], sr[2 * MT];                                    // (c_m, s_m) rotated by a quarter period
#pragma unroll
      for (int k = 0; k < 2 * MT; ++k) { cr[k] = sm[k]; sr[k] = -cm[k]; }
      auto series = [&](const double* image, auto sin_tag, const double (&c_)[2 * MT], const double (&s_)[2 * MT],
                        double (&acc)[4]) {
        constexpr bool SINP = decltype(sin_tag)::value;
        if (r_hi >= 0)
          mma_sweep<MT, KS, LdG, SINP>(image + (size_t)cell * RS, RS, r_lo, r_hi, off_w, wsrc, lane, q, AC, AS, AnC,
                                       AnS, c_, s_, acc);
        unsigned pd = pend0;
        while (pd) {
          const int i0L = __shfl_sync(0xffffffffu, i0, __ffs(pd) - 1);
          const bool mine = ingrp && outside && i0 == i0L;
          const int off_f = __shfl_sync(0xffffffffu, mine ? 0 : kMmaNone, src);
          mma_sweep<MT, KS, LdG, SINP>(image + (size_t)(i0L + 2) * RS, RS, 0, 3, off_f, wsrc, lane, q, AC, AS, AnC,
                                       AnS, c_, s_, acc);
          pd &= ~__ballot_sync(0xffffffffu, mine);
        }
      };
      if (f.mma_image_bs) series(f.mma_image_bs, std::true_type{}, cr, sr, o);
      if (f.mma_image_kc) series(f.mma_image_kc, std::false_type{}, cm, sm, ok);
      if (f.mma_image_ks) series(f.mma_image_ks, std::true_type{}, cr, sr, ok);
    }
    // ---- back to the particle lanes: lane 8 G + g takes the quad sum of fragment lanes 4 g .. 4 g + 3 ---------------
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const double v = __shfl_sync(0xffffffffu, quad_sum(o[k]), 4 * (lane & 7));
      if (ingrp) fb[k] = v;
    }
    if constexpr (EXTRA) {
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const double v = __shfl_sync(0xffffffffu, quad_sum(ok[k]), 4 * (lane & 7));
        if (ingrp) fk[k] = v;
      }
    }
  }
  // ---- particle role: profiles, perturbation, guiding-centre algebra ------------------------------------------------
  if (active) {
    const double* prow = inwin ? win + (size_t)off * RS : f.mma_image + (size_t)(i0 + 2) * RS;
    Profiles pr;
    double v[4];
#pragma unroll
    for (int a = 0; a < 4; ++a) v[a] = prow[(size_t)a * RS + R::kProf];
    pr.G = dot4(w, v); pr.Gs = dot4(dw, v);
#pragma unroll
    for (int a = 0; a < 4; ++a) v[a] = prow[(size_t)a * RS + R::kProf + 1];
    pr.I = dot4(w, v); pr.Is = dot4(dw, v);
#pragma unroll
    for (int a = 0; a < 4; ++a) v[a] = prow[(size_t)a * RS + R::kProf + 2];
    pr.io = dot4(w, v); pr.ios = dot4(dw, v);
    if constexpr (FIELD_ONLY) {
      dy[0] = fb[0]; dy[1] = fb[1]; dy[2] = fb[2]; dy[3] = fb[3] * (double)f.nfp;
      *prof_out = pr;
    } else {
    double pt[9];
#pragma unroll
    for (int k = 0; k < 9; ++k) pt[k] = 0.0;
    if constexpr (MODES) {
      const double zer = reduce_2pi(y[2]);
      const double GI = pr.G + pr.io * pr.I, GI_s = pr.Gs + pr.ios * pr.I + pr.io * pr.Is;
      const double invGI = 1.0 / GI, gig = GI_s * invGI;               // one division per right-hand side
#pragma unroll 1
      for (int k = 0; k < f.nk; ++k) {
#pragma unroll
        for (int a = 0; a < 4; ++a) v[a] = prow[(size_t)a * RS + R::kModes + k];
        const double ph = dot4(w, v), ph_s = dot4(dw, v);
        const double m = (double)__ldg(f.mode_m + k), n = (double)__ldg(f.mode_n + k);
        const double om = __ldg(f.omega + k);
        const double wt = reduce_2pi(om * t);
        double sn, cs;
        sincos_poly(fma(m, thr, fma(-n, zer, wt + __ldg(f.phase + k))), sn, cs);
        const double inv = __ldg(f.inv_omega + k) * invGI;             // 1 / (omega (G + iota I))
        const double Nk = fma(pr.io, m, -n);
        const double ah = -ph * Nk * inv;
        const double ah_s = -(ph_s * Nk + ph * pr.ios * m) * inv + ph * Nk * inv * gig;
        pt[0] = fma(ph, sn, pt[0]);
        pt[1] = fma(ph_s, sn, pt[1]);
        pt[2] = fma(m * ph, cs, pt[2]);
        pt[3] = fma(-n * ph, cs, pt[3]);
        pt[4] = fma(ah, sn, pt[4]);
        pt[5] = fma(ah_s, sn, pt[5]);
        pt[6] = fma(m * ah, cs, pt[6]);
        pt[7] = fma(-n * ah, cs, pt[7]);
        pt[8] = fma(om * ah, cs, pt[8]);
      }
      pt[1] *= f.inv_psi0;
      pt[5] *= f.inv_psi0;
    }
    fb[3] *= (double)f.nfp;
    if (EXTRA && (f.mma_image_kc || f.mma_image_ks)) {
      fk[3] *= (double)f.nfp;
      gc_algebra_general(mass, charge, mu, f.inv_psi0, y[3] * v_ref, fb, fk, pr, pt, dy);
    } else {
      gc_algebra(mass, charge, mu, f.inv_psi0, y[3] * v_ref, fb, pr, pt, dy);
    }
    dy[3] *= inv_v_ref;
    }
  }
}

// The table engine of trace_mma_kernel.
template <int MT, int KS, bool MODES, bool EXTRA = false>
struct MmaEngine {
  static constexpr bool kStageWindow = true;
  static __device__ __forceinline__ int win_doubles(const FieldDev& f) { return kMmaWinRows * f.mma_RS; }
  static constexpr int kExtDoubles = 2 * kMmaWtab;                   // per-thread weight table
  static __device__ __forceinline__ const double* win_src(const FieldDev& f, int cell) {
    return f.mma_image + (size_t)cell * f.mma_RS;                     // image rows cell .. cell+7
  }
  static __device__ __forceinline__ void rhs(const FieldDev& f, const double* win, double* ext, int cell, bool active,
                                             double mass, double charge, double mu, double v_ref, double inv_v_ref,
                                             double t, const double (&y)[4], double (&dy)[4]) {
    rhs_mma<MT, KS, MODES, EXTRA>(f, win, ext, cell, active, mass, charge, mu, v_ref, inv_v_ref, t, y, dy);
  }
  // B, B_s, B_theta, B_zeta and the profiles at (s, theta, zeta); must be called by all 32 lanes of a warp.
  static __device__ __forceinline__ void field(const FieldDev& f, const double* win, double* ext, int cell, bool active,
                                               double s, double th, double ze, double (&fb)[4], Profiles& pr) {
    const double y[4] = {s, th, ze, 0.0};
    rhs_mma<MT, KS, false, false, true>(f, win, ext, cell, active, 1.0, 1.0, 0.0, 1.0, 1.0, 0.0, y, fb, &pr);
  }
};

template <int MT, int KS, bool MODES, bool SAMPLE, bool EXTRA = false>
__global__ void __launch_bounds__(kMmaThreads, kMmaBlocksPerSm)
trace_mma_kernel(FieldDev f, TraceDev p, TileScratch sc, int mode, double* rhs_out) {
  trace_binned_body<MmaEngine<MT, KS, MODES, EXTRA>, kMmaThreads, kMmaCap, SAMPLE>(f, p, sc, mode, rhs_out);
}

// NEXT-3 on the direct harmonic sum: the symplectic explicit-implicit Euler integrator inside the same cell-binned
// persistent body (binning, tiles, record slots, DMMA sweep); every pass of a lane is one evaluation of the field, i.e.
// one quasi-Newton iteration of its current step (kernels_symplectic.cuh has the scheme).
template <int MT, int KS>
__global__ void __launch_bounds__(kMmaThreads, kMmaBlocksPerSm)
trace_mma_symplectic_kernel(FieldDev f, TraceDev p, TileScratch sc, int mode, double* rhs_out) {
  trace_binned_body<MmaEngine<MT, KS, false, false>, kMmaThreads, kMmaCap, false, 1>(f, p, sc, mode, rhs_out);
}

}  // namespace gc
