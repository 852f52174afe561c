// kernels_mma.cuh -- hot-path kernel for large ensembles, second generation: the harmonic sum as FP64 matrix
// instructions (DMMA.8x8x4), four lanes per particle.
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
// table, identical for the eight particles of a warp and fetched ONCE per warp (one 16-byte load per lane feeds
// four DMMA = 32 DFMA-equivalents per lane), the accumulators never leave registers.  On B200 DMMA.8x8x4 runs on
// the FP64 pipe at the DFMA rate (37 TFLOP/s measured, same roofline), so this buys operand bandwidth, not peak.
//
// Layout of the work.  A warp owns 8 particles; lane = 4 g + q: g = particle slot, q = lane of the quad.
//   * DMMA fragments: A[g][q], B[q][g], D[g][2q, 2q+1].  Toroidal numbers n = 4 j + q + 1 (k-step j), poloidal
//     numbers m = 1 + 8 T + (column) (m-tile T).  m = 0 and n = 0 are handled beside the DMMA (n = 0 initialises
//     the PC accumulator, m = 0 is a 16-term DFMA sum split over the quad).
//   * Rows: a warp sweeps the UNION of the stencil rows of its 8 particles (4 rows when they share a stencil,
//     5 when they straddle a node); a particle's weight for a row outside its own stencil is exactly 0, so its
//     result does not depend on who it shares the warp with.
//   * Per row the epilogue turns the eight accumulators of a lane into its share of B, B_s, B_theta, B_zeta with
//     (c_m, s_m) and the Lagrange weights; the quad sums by two butterfly shuffles at the end.
//   * The integrator is component-parallel: lane q carries component q of (s, theta, zeta, u) and of k1..k7; the
//     error norm is a quad reduction; every decision is taken identically by the four lanes.
// Window: the 8 node rows cell-2 .. cell+5 of a by-node image (contiguous in global memory, ONE bulk TMA copy per
// cell change); stencils that start further than 2 rows from the tile's cell are swept from global memory with the
// same instruction sequence (bit-identical results).  Binning, epochs, tiles, records: as in kernels_tile.cuh.
#pragma once
#include <cooperative_groups.h>

#include "device_math.cuh"
#include "field.cuh"
#include "kernels_generic.cuh"
#include "kernels_tile.cuh"      // TileScratch, record layout, mbarrier / bulk-copy helpers, home_bin, cDp*

namespace gc {

constexpr int kMmaThreads = 128;                 // 4 warps
constexpr int kMmaTile = kMmaThreads / 4;        // particles per tile
constexpr int kMmaCap = 32;                      // attempted steps per particle per chunk
constexpr int kMmaWinRows = 8;                   // node rows cell-2 .. cell+5
constexpr int kMmaModeSlots = 4;                 // mode harmonics per lane (nk <= 16)

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

struct MmaSums {
  double B, Bs, Bth, Bze;                        // this lane's share; Bze lacks the factor nfp
  double G, Gs, I, Is, io, ios;                  // complete on every lane
  double ph[kMmaModeSlots], phs[kMmaModeSlots];  // mode amplitudes k = q + 4 i (value, d/ds)
};

__device__ __forceinline__ double quad_sum(double v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  return v;
}
__device__ __forceinline__ double quad_get(double v, int lane, int c) {
  return __shfl_sync(0xffffffffu, v, (lane & ~3) | c);
}
__device__ __forceinline__ double quad_get_masked(double v, int lane, int c, unsigned mask) {
  return __shfl_sync(mask, v, (lane & ~3) | c);
}
__device__ __forceinline__ bool quad_all(bool pred, int lane) {
  const unsigned b = __ballot_sync(0xffffffffu, pred);
  return ((b >> (lane & ~3)) & 0xFu) == 0xFu;
}

// Sweep node rows r_lo .. r_hi (warp-uniform) of the image at `base` (row r at base + r RS).  `off` is the row of
// this lane's particle's first stencil node (any value outside [r_lo - 3, r_hi] gives weight 0 everywhere).
// Must be executed by all 32 lanes.
template <int MT, int KS, bool MODES, class Ld>
__device__ __forceinline__ void mma_sweep(const double* base, int RS, int r_lo, int r_hi, int off, int lane, int q,
                                          int nk, const double (&w)[4], const double (&dw)[4],
                                          const double (&AC)[KS], const double (&AS)[KS], const double (&AnC)[KS],
                                          const double (&AnS)[KS], const double (&cm)[2 * MT],
                                          const double (&sm)[2 * MT], MmaSums& o) {
  using R = MmaRow<MT, KS>;
#pragma unroll 1
  for (int r = r_lo; r <= r_hi; ++r) {
    const int idx = r - off;
    const double wr = idx == 0 ? w[0] : idx == 1 ? w[1] : idx == 2 ? w[2] : idx == 3 ? w[3] : 0.0;
    const double dwr = idx == 0 ? dw[0] : idx == 1 ? dw[1] : idx == 2 ? dw[2] : idx == 3 ? dw[3] : 0.0;
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
      const double m0 = (double)(1 + 8 * T + 2 * q), m1 = m0 + 1.0;
      const double c0 = cm[2 * T], s0 = sm[2 * T], c1 = cm[2 * T + 1], s1 = sm[2 * T + 1];
      T1 += fma(c0, PC0, s0 * QS0);
      T1 += fma(c1, PC1, s1 * QS1);
      T2 = fma(m0, fma(c0, QS0, -s0 * PC0), T2);
      T2 = fma(m1, fma(c1, QS1, -s1 * PC1), T2);
      T3 += fma(s0, QC0, -c0 * PS0);
      T3 += fma(s1, QC1, -c1 * PS1);
    }
    // m = 0: b(0,n) C_n and its zeta-derivative, n = 4 j + q + 1 on this lane; n = 0 on lane q = 0
    double x = (q == 0) ? Ld::ld1(row + R::kM0) : 0.0, xs = 0.0;
#pragma unroll
    for (int j = 0; j < KS; ++j) {
      const double b0 = Ld::ld1(row + R::kM0 + 1 + 4 * j + q);
      x = fma(b0, AC[j], x);
      xs = fma(b0, AnS[j], xs);
    }
    T1 += x;
    T3 -= xs;
    o.B = fma(wr, T1, o.B);
    o.Bs = fma(dwr, T1, o.Bs);
    o.Bth = fma(wr, T2, o.Bth);
    o.Bze = fma(wr, T3, o.Bze);
    const double g = Ld::ld1(row + R::kProf), ii = Ld::ld1(row + R::kProf + 1), io = Ld::ld1(row + R::kProf + 2);
    o.G = fma(wr, g, o.G);     o.Gs = fma(dwr, g, o.Gs);
    o.I = fma(wr, ii, o.I);    o.Is = fma(dwr, ii, o.Is);
    o.io = fma(wr, io, o.io);  o.ios = fma(dwr, io, o.ios);
    if constexpr (MODES) {
#pragma unroll
      for (int i = 0; i < kMmaModeSlots; ++i) {
        const int k = q + 4 * i;
        if (k < nk) {
          const double v = Ld::ld1(row + R::kModes + k);
          o.ph[i] = fma(wr, v, o.ph[i]);
          o.phs[i] = fma(dwr, v, o.phs[i]);
        }
      }
    }
  }
}

// Right-hand side, warp-collective: all 32 lanes call it; `on` is quad-uniform.  ysq = component q of the state
// at which to evaluate; returns component q of dy/dt (garbage for quads that are not on).
// win = shared-memory copy of image rows cell .. cell+7 (node rows cell-2 .. cell+5).
template <int MT, int KS, bool MODES>
__device__ __forceinline__ double rhs_mma(const FieldDev& f, const double* win, int cell, bool on, int lane, int q,
                                          double mass, double charge, double mu, double v_ref, double inv_v_ref,
                                          double t, double ysq) {
  double ys[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const double v = quad_get(ysq, lane, c);
    ys[c] = on ? v : 0.0;                                   // idle quads compute on zeros (finite operands)
  }
  int i0;
  double w[4], dw[4];
  lagrange_weights(f.ns, ys[0], i0, w, dw);
  const int off = i0 - cell + 2;
  const bool inwin = on && off >= 0 && off <= kMmaWinRows - 4;
  bool outside = on && !inwin;

  // ---- trigonometry: toroidal numbers n = 4 j + q + 1, poloidal numbers m = 1 + 8 T + 2 q + e ---------------------
  const double thr = reduce_2pi(ys[1]);
  const double phr = reduce_2pi((double)f.nfp * ys[2]);
  double AC[KS], AS[KS], AnC[KS], AnS[KS], cm[2 * MT], sm[2 * MT];
  sincos_poly((double)(q + 1) * phr, AS[0], AC[0]);
  {
    const double C4 = quad_get(AC[0], lane, 3), S4 = quad_get(AS[0], lane, 3);      // n = 4 lives on q = 3
#pragma unroll
    for (int j = 1; j < KS; ++j) {
      AC[j] = fma(AC[j - 1], C4, -AS[j - 1] * S4);
      AS[j] = fma(AS[j - 1], C4, AC[j - 1] * S4);
    }
#pragma unroll
    for (int j = 0; j < KS; ++j) {
      const double n = (double)(4 * j + q + 1);
      AnC[j] = n * AC[j];
      AnS[j] = n * AS[j];
    }
  }
  sincos_poly((double)(1 + 2 * q) * thr, sm[0], cm[0]);
  {
    const double c1 = quad_get(cm[0], lane, 0), s1 = quad_get(sm[0], lane, 0);      // m = 1 lives on q = 0
    cm[1] = fma(cm[0], c1, -sm[0] * s1);
    sm[1] = fma(sm[0], c1, cm[0] * s1);
    if constexpr (MT == 2) {
      const double c8 = quad_get(cm[1], lane, 3), s8 = quad_get(sm[1], lane, 3);    // m = 8 lives on q = 3
      cm[2] = fma(cm[0], c8, -sm[0] * s8);
      sm[2] = fma(sm[0], c8, cm[0] * s8);
      cm[3] = fma(cm[1], c8, -sm[1] * s8);
      sm[3] = fma(sm[1], c8, cm[1] * s8);
    }
  }

  MmaSums o;
  o.B = o.Bs = o.Bth = o.Bze = 0.0;
  o.G = o.Gs = o.I = o.Is = o.io = o.ios = 0.0;
#pragma unroll
  for (int i = 0; i < kMmaModeSlots; ++i) o.ph[i] = o.phs[i] = 0.0;
  const int RS = f.mma_RS;
  // ---- in-window stencils: one sweep over the union of their rows -----------------------------------------------
  const int r_lo = __reduce_min_sync(0xffffffffu, inwin ? off : 1 << 20);
  const int r_hi = __reduce_max_sync(0xffffffffu, inwin ? off + 3 : -1);
  if (r_hi >= 0)
    mma_sweep<MT, KS, MODES, LdS>(win, RS, r_lo, r_hi, inwin ? off : 1 << 20, lane, q, f.nk, w, dw, AC, AS, AnC, AnS,
                                  cm, sm, o);
  // ---- stencils outside the window: one sweep per distinct stencil, rows from global memory ------------------------
  unsigned pend = __ballot_sync(0xffffffffu, outside);
  while (pend) {
    const int leader = __ffs(pend) - 1;
    const int i0L = __shfl_sync(0xffffffffu, i0, leader);
    const bool mine = outside && i0 == i0L;
    mma_sweep<MT, KS, MODES, LdG>(f.mma_image + (size_t)(i0L + 2) * RS, RS, 0, 3, mine ? 0 : 1 << 20, lane, q, f.nk, w,
                                  dw, AC, AS, AnC, AnS, cm, sm, o);
    outside = outside && !mine;
    pend = __ballot_sync(0xffffffffu, outside);
  }
  const double fb[4] = {quad_sum(o.B), quad_sum(o.Bs), quad_sum(o.Bth), quad_sum(o.Bze) * (double)f.nfp};
  Profiles pr;
  pr.G = o.G; pr.Gs = o.Gs; pr.I = o.I; pr.Is = o.Is; pr.io = o.io; pr.ios = o.ios;
  double pt[9];
#pragma unroll
  for (int k = 0; k < 9; ++k) pt[k] = 0.0;
  if constexpr (MODES) {
    const double zer = reduce_2pi(ys[2]);
    const double GI = pr.G + pr.io * pr.I, GI_s = pr.Gs + pr.ios * pr.I + pr.io * pr.Is;
#pragma unroll
    for (int i = 0; i < kMmaModeSlots; ++i) {
      const int k = q + 4 * i;
      if (k < f.nk) {
        const double ph = o.ph[i], ph_s = o.phs[i];
        const double m = (double)__ldg(f.mode_m + k), n = (double)__ldg(f.mode_n + k);
        const double om = __ldg(f.omega + k);
        const double wt = reduce_2pi(om * t);
        double sn, cs;
        sincos_poly(fma(m, thr, fma(-n, zer, wt + __ldg(f.phase + k))), sn, cs);
        const double inv = 1.0 / (om * GI);
        const double Nk = fma(pr.io, m, -n);
        const double ah = -ph * Nk * inv;
        const double ah_s = -(ph_s * Nk + ph * pr.ios * m) * inv + ph * Nk * inv * (GI_s / GI);
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
    }
#pragma unroll
    for (int k = 0; k < 9; ++k) pt[k] = quad_sum(pt[k]);
    pt[1] *= f.inv_psi0;
    pt[5] *= f.inv_psi0;
  }
  double dy[4];
  gc_algebra(mass, charge, mu, f.inv_psi0, ys[3] * v_ref, fb, pr, pt, dy);
  dy[3] *= inv_v_ref;
  return q == 0 ? dy[0] : q == 1 ? dy[1] : q == 2 ? dy[2] : dy[3];
}

extern __shared__ __align__(128) unsigned char gc_mma_smem[];

// Dynamic shared memory of one block: window, stage derivatives, Poincare staging, barrier, tile id.
__host__ __device__ inline size_t mma_smem_bytes(int RS) {
  return (size_t)kMmaWinRows * RS * sizeof(double) + (size_t)7 * kMmaThreads * sizeof(double) +
         (size_t)kMmaTile * 16 * sizeof(double) + 64;
}

// mode 0: trace.  mode 1: right-hand side only (gc_rhs_eval): k1 of every particle goes to rhs_out[4][n].
template <int MT, int KS, bool MODES>
__global__ void __launch_bounds__(kMmaThreads, 2)
trace_mma_kernel(FieldDev f, TraceDev p, TileScratch sc, int mode, double* rhs_out) {
  cgx::grid_group grid = cgx::this_grid();
  const int tid = threadIdx.x;
  const int lane = tid & 31, q = tid & 3, slot = tid >> 2;
  const unsigned quadmask = 0xFu << (lane & ~3);
  const long long gtid = (long long)blockIdx.x * kMmaThreads + tid;
  const long long gthreads = (long long)gridDim.x * kMmaThreads;
  const int ncell = f.ns - 3;
  const int RS = f.mma_RS;
  constexpr double kTwoPi = 6.283185307179586476925286766559;

  double* win = reinterpret_cast<double*>(gc_mma_smem);                  // [8 RS]
  double* kbuf = win + kMmaWinRows * RS;                                 // [7][kMmaThreads]
  double* pbuf = kbuf + 7 * kMmaThreads;                                 // [kMmaTile][16]: dense-output coefficients
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(pbuf + kMmaTile * 16);
  int* s_int = reinterpret_cast<int*>(bar + 1);
  auto kb = [&](int j) -> double& { return kbuf[j * kMmaThreads + tid]; };

  if (tid == 0) mbar_init(bar, 1);
  __syncthreads();
  unsigned bar_phase = 0;

  // ---- P0: records from the inputs (coalesced), first bin counts ---------------------------------------------------
  for (long long i = gtid; i < p.n; i += gthreads) {
    double* r = sc.rec + i * kRecDoubles;
    int st = kStRunning;
    double y0, y1, y2, y3, h, t = p.t0, mu = p.mu[i];
    if (mode == 1) {
      y0 = p.s0[i]; y1 = p.th0[i]; y2 = p.ze0[i]; y3 = p.vpar0[i]; h = 0.0;
    } else {
      if (p.resume && p.status[i] != 0) st = kStSkip;
      y0 = p.s0[i]; y1 = p.th0[i]; y2 = p.ze0[i]; y3 = p.vpar0[i] * p.inv_v_ref;
      h = (p.h_inout && p.h_inout[i] > 0.0) ? p.h_inout[i] : p.h0;
      if (h < p.h_min) h = p.h_min;
    }
    const int bin = home_bin(f.ns, y0);
    reinterpret_cast<double4*>(r)[0] = make_double4(y0, y1, y2, y3);
    reinterpret_cast<double4*>(r)[1] = make_double4(0.0, 0.0, 0.0, 0.0);
    reinterpret_cast<double4*>(r)[2] = make_double4(t, h, mu, __longlong_as_double(0LL));
    int4 a = make_int4(st, 0, 0, 0), b = make_int4(0, bin, 0, 0);
    reinterpret_cast<int4*>(r + 12)[0] = a;
    reinterpret_cast<int4*>(r + 12)[1] = b;
    if (st == kStRunning) atomicAdd(sc.cnt + bin, 1);
  }
  grid.sync();

  for (;;) {
    // ---- B: segment and tile offsets (block 0) -------------------------------------------------------------------
    if (blockIdx.x == 0) {
      int* wsp = reinterpret_cast<int*>(win);                            // nbin + 2 ncell ints staged in the window space
      const int nbin = ncell * kSubBins;
      for (int b = tid; b < nbin; b += kMmaThreads) { wsp[b] = __ldcg(sc.cnt + b); sc.cnt[b] = 0; }
      __syncthreads();
      if (tid == 0) {
        int run = 0, tiles = 0;
        for (int c = 0; c < ncell; ++c) {
          wsp[nbin + c] = run;
          wsp[nbin + ncell + c] = tiles;
          const int run0 = run;
          for (int b = c * kSubBins; b < (c + 1) * kSubBins; ++b) {
            const int k = wsp[b];
            wsp[b] = run;
            run += k;
          }
          tiles += (run - run0 + kMmaTile - 1) / kMmaTile;
        }
        sc.start[ncell] = run;
        sc.tstart[ncell] = tiles;
        sc.ctrl[0] = 0; sc.ctrl[1] = 0; sc.ctrl[2] = tiles; sc.ctrl[3] = run;
      }
      __syncthreads();
      for (int b = tid; b < nbin; b += kMmaThreads) sc.cursor[b] = wsp[b];
      for (int c = tid; c < ncell; c += kMmaThreads) {
        sc.start[c] = wsp[nbin + c];
        sc.tstart[c] = wsp[nbin + ncell + c];
      }
      __syncthreads();
    }
    grid.sync();
    const int ntiles = __ldcg(sc.ctrl + 2);
    if (__ldcg(sc.ctrl + 3) == 0) break;

    // ---- C: scatter the running particles into bin order -----------------------------------------------------------
    for (long long i = gtid; i < p.n; i += gthreads) {
      const int2 sf = __ldcg(reinterpret_cast<const int2*>(sc.rec + i * kRecDoubles + 12));
      if (sf.x == kStRunning) {
        const int bin = __ldcg(reinterpret_cast<const int2*>(sc.rec + i * kRecDoubles + 14)).y;
        sc.order[atomicAdd(sc.cursor + bin, 1)] = (int)i;
      }
    }
    grid.sync();

    // ---- D: tiles ------------------------------------------------------------------------------------------------
    int cur_cell = -1;
    __syncthreads();
    if (tid == 0) s_int[0] = atomicAdd(sc.ctrl + 0, 1);
    __syncthreads();
    for (;;) {
      const int tile = s_int[0];                                         // grabbed before the loop / at chunk end
      if (tile >= ntiles) break;
      int lo = 0, hi = ncell - 1;                                        // largest c with tstart[c] <= tile
      while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (__ldcg(sc.tstart + mid) <= tile) lo = mid; else hi = mid - 1;
      }
      const int cell = lo;
      const int seg0 = __ldcg(sc.start + cell), seg1 = __ldcg(sc.start + cell + 1);
      const int begin = seg0 + (tile - __ldcg(sc.tstart + cell)) * kMmaTile;
      const int count = min(kMmaTile, seg1 - begin);
      if (cell != cur_cell) {                                            // stage the window: one bulk copy
        if (tid == 0) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          const unsigned bytes = (unsigned)(kMmaWinRows * RS * sizeof(double));
          mbar_expect_tx(bar, bytes);
          bulk_g2s(win, f.mma_image + (size_t)cell * RS, bytes, bar);    // image rows cell .. cell+7 = nodes cell-2 .. cell+5
        }
        mbar_wait(bar, bar_phase);
        bar_phase ^= 1u;
        cur_cell = cell;
      }

      // quad state: every lane of a quad carries the particle's scalars; lane q carries component q of y
      const bool active = slot < count;
      long long pid = 0;
      double yq = 0.0, ynq = 0.0, t = 0.0, h = 0.0, mu = 0.0;
      long long attempts = 0;
      int st = 0, flags = 0, n_acc = 0, n_rej = 0, n_forced = 0;
      kb(0) = 0.0;
      if (active) {
        pid = __ldcg(sc.order + begin + slot);
        const double* r = sc.rec + pid * kRecDoubles;
        yq = __ldcg(r + q);
        kb(0) = __ldcg(r + 4 + q);
        const double4 c = ldcg4(r + 8);
        const int4 d = __ldcg(reinterpret_cast<const int4*>(r + 12));
        const int4 g = __ldcg(reinterpret_cast<const int4*>(r + 12) + 1);
        t = c.x; h = c.y; mu = c.z; attempts = __double_as_longlong(c.w);
        st = d.x; flags = d.y; n_acc = d.z; n_rej = d.w; n_forced = g.x;
      }
      bool running = active;                     // false once finished or parked
      bool first_chunk = true;
      bool extra = false;                        // an extra chunk: stop as soon as the epoch's first chunks are done

      for (;;) {                                 // chunks of kMmaCap attempts
#pragma unroll 1
        for (int att = 0; att < kMmaCap; ++att) {
          if (!__any_sync(0xffffffffu, running)) break;
          if (extra) {                           // attempts are warp-local: any warp may stop at any attempt
            int done = 0;
            if (lane == 0) done = *reinterpret_cast<const volatile int*>(sc.ctrl + 1);
            if (__shfl_sync(0xffffffffu, done, 0) >= ntiles) break;
          }
          const bool do_k1 = __any_sync(0xffffffffu, running && !(flags & kFlagHaveK1));
          double h_try = h;
          bool clipped = false;
          const bool forced = (flags & kFlagPrevRejected) && p.h_min > 0.0 && h == p.h_min;
          if (mode == 0 && running && t < p.t_max) {
            if (t + h_try >= p.t_max) { h_try = p.t_max - t; clipped = true; }
            if (!(t + h_try > t)) { st = GC_ST_NONFINITE_; running = false; }       // step underflow
          }
          ynq = yq;
#pragma unroll 1
          for (int stage = do_k1 ? 0 : 1; stage <= 6; ++stage) {
            if (stage > 0 && !__any_sync(0xffffffffu, running)) break;
            double ysq, ts;
            if (stage == 0) {
              ysq = yq;
              ts = t;
            } else {
              double acc = 0.0;
              for (int j = 0; j < stage; ++j) acc = fma(cDpA[stage][j], kb(j), acc);
              ysq = fma(h_try, acc, yq);
              ts = fma(cDpC[stage], h_try, t);
              if (stage == 6) ynq = ysq;
            }
            const bool lane_on = running && (stage > 0 || !(flags & kFlagHaveK1));
            const double dyq = rhs_mma<MT, KS, MODES>(f, win, cell, lane_on, lane, q, p.mass, p.charge, mu, p.v_ref,
                                                     p.inv_v_ref, ts, ysq);
            if (lane_on) kb(stage) = dyq;
            if (stage == 0) {
              const bool fin = quad_all(isfinite(yq) && isfinite(dyq), lane);
              if (lane_on) {
                flags |= kFlagHaveK1;
                if (mode == 1) {
                  rhs_out[(long long)q * p.n + pid] = dyq;
                  st = 0; running = false;
                } else if (!fin) {
                  st = GC_ST_NONFINITE_; running = false;
                } else if (!(t < p.t_max)) {
                  st = 0; running = false;
                }
              }
            }
          }
          // error norm and neighbours' components: warp-collective, executed by every lane
          double e = 0.0;
          for (int j = 0; j < 7; ++j) e = fma(cDpE[j], kb(j), e);
          const double delta = h_try * e;
          const double sk = fma(p.rtol, fmax(fabs(yq), fabs(ynq)), p.atol);
          const double rr = delta / sk;
          const double err = sqrt(quad_sum(rr * rr) * 0.25);
          const bool finq = quad_all(isfinite(ynq) && isfinite(kb(6)), lane);
          const double s_new = quad_get(ynq, lane, 0);
          const double ze_old = quad_get(yq, lane, 2), ze_new = quad_get(ynq, lane, 2);
          if (running) {
            ++attempts;
            const bool finite = finq && isfinite(err);
            bool accept;
            if (forced) {
              accept = finite;
              if (!finite) { st = GC_ST_NONFINITE_; running = false; }
            } else {
              accept = finite && err <= 1.0;
            }
            if (running && accept) {
              const double scl = scale_after_accept(err);
              const double h_next = (flags & kFlagPrevRejected) ? h_try * fmin(scl, 1.0) : h_try * scl;
              if (p.poincare_capacity > 0 && floor(ze_old / kTwoPi) != floor(ze_new / kTwoPi)) {
                // dense-output coefficients of component q -> pbuf; lane 0 of the quad locates the crossings
                if (q < 3) {
                  double dd = 0.0;
                  for (int j = 0; j < 7; ++j) dd = fma(cDpD[j], kb(j), dd);
                  const double r2 = ynq - yq, r3 = h_try * kb(0) - r2, r4 = r2 - h_try * kb(6) - r3;
                  double* pb = pbuf + slot * 16 + q * 5;
                  pb[0] = yq; pb[1] = r2; pb[2] = r3; pb[3] = r4; pb[4] = h_try * dd;
                }
                __syncwarp(quadmask);
                if (q == 0) {
                  Dense3 d;
                  const double* pb = pbuf + slot * 16;
#pragma unroll
                  for (int c = 0; c < 3; ++c) {
                    d.r1[c] = pb[c * 5]; d.r2[c] = pb[c * 5 + 1]; d.r3[c] = pb[c * 5 + 2];
                    d.r4[c] = pb[c * 5 + 3]; d.r5[c] = pb[c * 5 + 4];
                  }
                  poincare_emit(d, pid, t, h_try, ze_old, ze_new, p.poincare, p.poincare_capacity, p.poincare_count);
                }
                __syncwarp(quadmask);
              }
              t = clipped ? p.t_max : t + h_try;
              yq = ynq;
              kb(0) = kb(6);
              ++n_acc;
              if (forced) ++n_forced;
              flags &= ~kFlagPrevRejected;
              if (!clipped) h = h_next;
              if (h < p.h_min) h = p.h_min;
              if (s_new >= p.s_loss) st = 1;
              else if (s_new <= p.s_min) st = 2;
              else if (clipped) st = 0;
              else if (attempts >= p.max_steps) st = 3;
              if (st != kStRunning) running = false;
              else {
                const int hc = home_cell(f.ns, s_new);
                if (hc < cell - 1 || hc > cell + 1) running = false;      // parked until the next binning
              }
            } else if (running) {
              ++n_rej;
              h = h_try * scale_after_reject(err);
              if (h < p.h_min) h = p.h_min;
              flags |= kFlagPrevRejected;
              if (attempts >= p.max_steps) { st = 3; running = false; }
            }
          }
        }
        // chunk end: take the next tile if there is one; if the epoch's tiles are all handed out, keep
        // advancing this one while other blocks still work on a first chunk (no idle tail)
        if (first_chunk && tid == 0) atomicAdd(sc.ctrl + 1, 1);
        first_chunk = false;
        const int nrun = __syncthreads_count(running);
        if (tid == 0) {
          const int next = atomicAdd(sc.ctrl + 0, 1);
          bool more = false;
          if (next >= ntiles && nrun * 2 >= kMmaThreads) {
            const volatile int* vc = sc.ctrl;
            more = vc[1] < ntiles;
          }
          s_int[0] = next;
          s_int[1] = more;
        }
        __syncthreads();
        if (!s_int[1]) break;
        extra = true;
      }
      // write the tile back
      if (active) {
        double* r = sc.rec + pid * kRecDoubles;
        const double s_now = quad_get_masked(yq, lane, 0, quadmask);
        __stcg(r + q, yq);
        __stcg(r + 4 + q, kb(0));
        if (q == 0) {
          const int hb = home_bin(f.ns, s_now);
          stcg4(r + 8, make_double4(t, h, mu, __longlong_as_double(attempts)));
          __stcg(reinterpret_cast<int4*>(r + 12), make_int4(st, flags, n_acc, n_rej));
          __stcg(reinterpret_cast<int4*>(r + 12) + 1, make_int4(n_forced, hb, 0, 0));
          if (st == kStRunning) atomicAdd(sc.cnt + hb, 1);
        }
      }
      __syncthreads();                                                   // window / kbuf / s_int are reused
    }
    grid.sync();
  }

  // ---- outputs (coalesced) -------------------------------------------------------------------------------------
  if (mode == 0) {
    for (long long i = gtid; i < p.n; i += gthreads) {
      const double* r = sc.rec + i * kRecDoubles;
      const int4 d = __ldcg(reinterpret_cast<const int4*>(r + 12));
      if (d.x == kStSkip) continue;
      const double4 a = ldcg4(r);
      const double4 c = ldcg4(r + 8);
      const int n_forced = __ldcg(reinterpret_cast<const int4*>(r + 12) + 1).x;
      p.y_out[i] = a.x;
      p.y_out[p.n + i] = a.y;
      p.y_out[2 * p.n + i] = a.z;
      p.y_out[3 * p.n + i] = a.w * p.v_ref;
      p.t_out[i] = c.x;
      p.status[i] = d.x;
      if (p.h_inout) p.h_inout[i] = c.y;
      if (p.n_acc) p.n_acc[i] = (p.resume ? p.n_acc[i] : 0) + d.z;
      if (p.n_rej) p.n_rej[i] = (p.resume ? p.n_rej[i] : 0) + d.w;
      if (p.n_forced) p.n_forced[i] = (p.resume ? p.n_forced[i] : 0) + n_forced;
    }
  }
}

}  // namespace gc
