// kernels_tile.cuh -- the hot-path kernel for large ensembles: persistent, cell-binned, one THREAD per particle.
//
// Idea.  The radial stencil of a right-hand side depends only on the particle's radial
// cell, and thousands of particles share a cell.  Particles are therefore binned by the start i0 of their
// stencil ("home cell"); a block of 128 threads takes a TILE of up to 128 particles of one cell, stages that
// cell's window of the harmonic table -- the six node rows i0-1 .. i0+4, i.e. the home stencil and both
// neighbours -- into shared memory with ONE bulk (TMA) copy of a pre-packed image, and every thread then
// integrates its own particle: the table values it needs are the same address for (almost) all lanes of a
// warp, so a shared-memory load is a broadcast, and everything that is per particle (Lagrange weights, the two
// sincos, the angle-addition recurrences, the guiding-centre algebra, the Dormand-Prince controller) is done
// by one lane instead of being replicated over a warp.
//
// Radial interpolation commutes with the harmonic sum, so the inner loop carries none: with
//     b(m,n) cos(m th - n ph) + b(m,-n) cos(m th + n ph) = P c_m C_n + Q s_m S_n      (ph = nfp zeta)
// a thread accumulates, per poloidal row m and per stencil slot a = 0..3,
//     PC[a] += P[a] C_n,  PS[a] += P[a] n S_n,  QS[a] += Q[a] S_n,  QC[a] += Q[a] n C_n
// (16 DFMA + 2 DMUL per (m,n) pair against four 16-byte broadcast loads) and applies the four Lagrange
// weights and (c_m, s_m) once per row.  C_n, S_n come from one sincos(nfp zeta) by recurrence and stay in
// registers; c_m, s_m advance by the same recurrence from one sincos(theta) as the rows go by.
//
// Work distribution.  One cooperative persistent launch per gc_trace call.  Each epoch: block 0 turns the
// per-cell counts into segment offsets, all threads scatter the running particles into `order`, blocks pull
// tiles through an atomic counter and give every lane up to kTileCap attempted steps.  A lane whose particle
// finishes, or whose home cell moves more than one cell away from the tile's, idles until the tile is written
// back; a stage that needs a row outside the window reads the same image from global memory (identical
// arithmetic, so a particle's result does not depend on who it shared a tile with).  Blocks that run out of
// tiles keep advancing the tile they hold until every tile of the epoch has had its first chunk, so an epoch
// has no idle tail.  Finished and lost particles simply stop being binned: that is the compaction.
#pragma once
#include <cooperative_groups.h>

#include "device_math.cuh"
#include "field.cuh"
#include "kernels_generic.cuh"   // Profiles, gc_algebra, Dense3, poincare_emit

namespace gc {

namespace cgx = cooperative_groups;

constexpr int kTileThreads = 128;      // tile kernel: particles per tile = threads per block
#ifndef GC_TILE_CAP
#define GC_TILE_CAP 8
#endif
constexpr int kTileCap = GC_TILE_CAP;  // tile kernel: attempted steps per lane per chunk
constexpr int kRecDoubles = 16;        // one 128-byte record per particle
#ifndef GC_SUBBINS
#define GC_SUBBINS 8
#endif
constexpr int kSubBins = GC_SUBBINS;   // radial sub-bins per cell: tiles come out ordered in s (lane coherence)

// Per-call scratch of the tile kernel (device memory, owned by gc_trace for the duration of the call).
struct TileScratch {
  double* rec;      // [slots][16]: y[4], k1[4], t, h, mu, attempts (int64), {status, flags, n_acc, n_rej}, {n_forced, bin, jn, particle}
  int* order;       // [slots] slots of the running particles sorted by home cell
  int* cnt;         // [ncell kSubBins] running particles per bin (home cell, radial sub-bin), for the NEXT binning
  int* start;       // [ncell + 1] cell segment offsets into order
  int* tstart;      // [ncell + 1] tile offsets
  int* cursor;      // [ncell kSubBins] scatter cursors
  int tile_size;    // particles per tile, a multiple of 8, <= threads per block
  int chunk;        // attempted steps per lane per chunk (<= the kernel's CAP template argument: 0 = CAP)
  long long slots;  // record slots: the ensemble streams through them inside one launch -- a slot whose particle has
                    // finished is flushed to the outputs and handed to the next unstarted particle -- so that the
                    // records stay in L2 between epochs (10^6 records of 128 B do not fit)
  unsigned long long* next;   // input cursor: first particle not yet admitted
  int* ctrl;        // [0] tile counter, [1] tiles past their first chunk, [2] tiles this epoch, [3] running, [4] input exhausted
};

enum { kFlagPrevRejected = 1, kFlagHaveK1 = 2, kFlagFresh = 4, kFlagFinal = 8 };   // 4, 8: symplectic passes
enum { kStRunning = -1, kStSkip = -2, kStEmpty = -3 };   // slot states below 0; >= 0: finished, not yet flushed

__constant__ double cDpA[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {dp::a21, 0, 0, 0, 0, 0},
    {dp::a31, dp::a32, 0, 0, 0, 0},
    {dp::a41, dp::a42, dp::a43, 0, 0, 0},
    {dp::a51, dp::a52, dp::a53, dp::a54, 0, 0},
    {dp::a61, dp::a62, dp::a63, dp::a64, dp::a65, 0},
    {dp::a71, 0.0, dp::a73, dp::a74, dp::a75, dp::a76}};
__constant__ double cDpC[7] = {0.0, dp::c2, dp::c3, dp::c4, dp::c5, 1.0, 1.0};
__constant__ double cDpE[7] = {dp::e1, 0.0, dp::e3, dp::e4, dp::e5, dp::e6, dp::e7};
__constant__ double cDpD[7] = {dp::d1, 0.0, dp::d3, dp::d4, dp::d5, dp::d6, dp::d7};

// ---- mbarrier / bulk-copy primitives (sm_90+ PTX; SASS: SYNCS / UBLKCP) ------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

// ---- loaders: four stencil values of one table entry -------------------------------------------------------------
struct LdShared {
  static __device__ __forceinline__ void ld4(const double* p, double (&v)[4]) {
    const double2 a = *reinterpret_cast<const double2*>(p);
    const double2 b = *reinterpret_cast<const double2*>(p + 2);
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
  }
};
struct LdGlobal {
  static __device__ __forceinline__ void ld4(const double* p, double (&v)[4]) {
    const double2 a = __ldg(reinterpret_cast<const double2*>(p));
    const double2 b = __ldg(reinterpret_cast<const double2*>(p + 2));
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
  }
};

__device__ __forceinline__ double dot4(const double (&w)[4], const double (&v)[4]) {
  return fma(w[3], v[3], fma(w[2], v[2], fma(w[1], v[1], w[0] * v[0])));
}

// Field quantities one right-hand side needs, as they come out of the table sweep.
struct TileSums {
  double B, Bs, Bth, Bze;       // Bze still lacks the factor nfp
  Profiles pr;
  double pt[9];                 // perturbation block (raw: psi-derivatives still d/ds)
};

// One sweep over the table entries of a stencil: rows m = 0..M of [b(m,0), (P,Q)(m,1), ..., (P,Q)(m,NMAX)], then
// G, I, iota, then the mode amplitudes.  `e` points at the lane's first stencil value of entry 0; consecutive
// entries are `stride` doubles apart.
template <int NMAX, bool MODES, class Ld>
__device__ __forceinline__ void table_sweep(const FieldDev& f, const double* e, int stride, const double (&w)[4],
                                            const double (&dw)[4], double c1, double s1, const double (&C)[NMAX + 1],
                                            const double (&S)[NMAX + 1], double thr, double zer, double t,
                                            TileSums& o) {
  double B = 0.0, Bs = 0.0, Bth = 0.0, Bze = 0.0;
  double cm = 1.0, sm = 0.0;
  const int M = f.M;
#pragma unroll 1
  for (int m = 0; m <= M; ++m) {
    double PC[4], PS[4] = {0.0, 0.0, 0.0, 0.0}, QS[4] = {0.0, 0.0, 0.0, 0.0}, QC[4] = {0.0, 0.0, 0.0, 0.0};
    Ld::ld4(e, PC);                                        // n = 0 column
    e += stride;
#pragma unroll
    for (int n = 1; n <= NMAX; ++n) {
      double P[4], Q[4];
      Ld::ld4(e, P);
      Ld::ld4(e + stride, Q);
      e += 2 * stride;
      const double nS = (double)n * S[n], nC = (double)n * C[n];
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        PC[a] = fma(P[a], C[n], PC[a]);
        PS[a] = fma(P[a], nS, PS[a]);
        QS[a] = fma(Q[a], S[n], QS[a]);
        QC[a] = fma(Q[a], nC, QC[a]);
      }
    }
    const double pc = dot4(w, PC), pcs = dot4(dw, PC), qs = dot4(w, QS), qss = dot4(dw, QS);
    const double ps = dot4(w, PS), qc = dot4(w, QC);
    B = fma(cm, pc, fma(sm, qs, B));
    Bs = fma(cm, pcs, fma(sm, qss, Bs));
    Bth = fma((double)m, fma(cm, qs, -sm * pc), Bth);
    Bze = fma(sm, qc, fma(-cm, ps, Bze));
    const double cn = fma(cm, c1, -sm * s1);
    sm = fma(sm, c1, cm * s1);
    cm = cn;
  }
  o.B = B; o.Bs = Bs; o.Bth = Bth; o.Bze = Bze;
  double v[4];
  Ld::ld4(e, v); o.pr.G = dot4(w, v); o.pr.Gs = dot4(dw, v); e += stride;
  Ld::ld4(e, v); o.pr.I = dot4(w, v); o.pr.Is = dot4(dw, v); e += stride;
  Ld::ld4(e, v); o.pr.io = dot4(w, v); o.pr.ios = dot4(dw, v); e += stride;
#pragma unroll
  for (int q = 0; q < 9; ++q) o.pt[q] = 0.0;
  if constexpr (MODES) {
    const Profiles& p = o.pr;
    const double GI = p.G + p.io * p.I, GI_s = p.Gs + p.ios * p.I + p.io * p.Is;
#pragma unroll 1
    for (int k = 0; k < f.nk; ++k) {
      Ld::ld4(e, v);
      e += stride;
      const double ph = dot4(w, v), ph_s = dot4(dw, v);
      const double m = (double)__ldg(f.mode_m + k), n = (double)__ldg(f.mode_n + k);
      const double om = __ldg(f.omega + k);
      const double wt = reduce_2pi(om * t);
      double sn, cs;
      sincos_poly(fma(m, thr, fma(-n, zer, wt + __ldg(f.phase + k))), sn, cs);
      const double inv = 1.0 / (om * GI);
      const double Nk = fma(p.io, m, -n);
      const double ah = -ph * Nk * inv;
      const double ah_s = -(ph_s * Nk + ph * p.ios * m) * inv + ph * Nk * inv * (GI_s / GI);
      o.pt[0] = fma(ph, sn, o.pt[0]);
      o.pt[1] = fma(ph_s, sn, o.pt[1]);
      o.pt[2] = fma(m * ph, cs, o.pt[2]);
      o.pt[3] = fma(-n * ph, cs, o.pt[3]);
      o.pt[4] = fma(ah, sn, o.pt[4]);
      o.pt[5] = fma(ah_s, sn, o.pt[5]);
      o.pt[6] = fma(m * ah, cs, o.pt[6]);
      o.pt[7] = fma(-n * ah, cs, o.pt[7]);
      o.pt[8] = fma(om * ah, cs, o.pt[8]);
    }
  }
}

// Right-hand side of one lane.  win = shared-memory image of the tile's cell ([E][6] rows cell-1..cell+4, then
// [E][4] rows cell..cell+3); lanes whose stencil is not in the window read their own cell's image from global
// memory.  Must be called by all 32 lanes of a warp; inactive lanes do nothing.
template <int NMAX, bool MODES>
__device__ __forceinline__ void rhs_tile(const FieldDev& f, const double* win, int cell, bool active, double mass,
                                         double charge, double mu, double v_ref, double inv_v_ref, double t,
                                         const double (&y)[4], double (&dy)[4]) {
  int i0;
  double w[4], dw[4];
  lagrange_weights(f.ns, y[0], i0, w, dw);
  const int off = i0 - cell + 1;
  const bool inwin = active && off >= 0 && off <= 2;
  const bool outside = active && !inwin;
  const double thr = reduce_2pi(y[1]);
  const double phr = reduce_2pi((double)f.nfp * y[2]);
  double c1, s1, C[NMAX + 1], S[NMAX + 1];
  sincos_poly(thr, s1, c1);
  sincos_poly(phr, S[1], C[1]);
  C[0] = 1.0; S[0] = 0.0;
#pragma unroll
  for (int n = 2; n <= NMAX; ++n) {
    C[n] = fma(C[n - 1], C[1], -S[n - 1] * S[1]);
    S[n] = fma(S[n - 1], C[1], C[n - 1] * S[1]);
  }
  const double zer = MODES ? reduce_2pi(y[2]) : 0.0;
  TileSums o;
  const int E = f.tile_E;
  if (inwin) {
    const double* e = (off == 1) ? win + 6 * E : win + off;     // off = 0 or 2: rows 0..3 or 2..5 of [E][6]
    table_sweep<NMAX, MODES, LdShared>(f, e, off == 1 ? 4 : 6, w, dw, c1, s1, C, S, thr, zer, t, o);
  }
  if (__any_sync(0xffffffffu, outside)) {
    if (outside) {
      const double* e = f.tile_images + (size_t)i0 * (10 * E) + 6 * E;
      table_sweep<NMAX, MODES, LdGlobal>(f, e, 4, w, dw, c1, s1, C, S, thr, zer, t, o);
    }
  }
  if (active) {
    const double fb[4] = {o.B, o.Bs, o.Bth, o.Bze * (double)f.nfp};
    o.pt[1] *= f.inv_psi0;
    o.pt[5] *= f.inv_psi0;
    gc_algebra(mass, charge, mu, f.inv_psi0, y[3] * v_ref, fb, o.pr, o.pt, dy);
    dy[3] *= inv_v_ref;
  }
}

// L2-coherent 32-byte record accesses (the scratch is written by other blocks during the launch: bypass L1)
__device__ __forceinline__ double4 ldcg4(const double* p) {
  const double2 a = __ldcg(reinterpret_cast<const double2*>(p));
  const double2 b = __ldcg(reinterpret_cast<const double2*>(p) + 1);
  return make_double4(a.x, a.y, b.x, b.y);
}
__device__ __forceinline__ void stcg4(double* p, double4 v) {
  __stcg(reinterpret_cast<double2*>(p), make_double2(v.x, v.y));
  __stcg(reinterpret_cast<double2*>(p) + 1, make_double2(v.z, v.w));
}

__device__ __forceinline__ int home_cell(int ns, double s) { return stencil_start(ns, s * (double)(ns - 1)); }

// Bin = home cell * kSubBins + radial sub-bin.  The sub-bin only orders the particles of a cell by s, so that
// neighbouring lanes of a tile use the same stencil offset most of the time (shared-memory loads of a lane pair
// merge when both read the same 16 bytes); it has no influence on any particle's arithmetic.
__device__ __forceinline__ int home_bin(int ns, double s) {
  const double u = s * (double)(ns - 1);
  const int cell = stencil_start(ns, u);
  double fr = (u - (double)(cell + 1)) * (double)kSubBins;          // interior: u in [cell + 1, cell + 2)
  int sub = fr >= 0.0 ? (fr < (double)kSubBins ? (int)fr : kSubBins - 1) : 0;   // NaN -> 0
  return cell * kSubBins + sub;
}

extern __shared__ __align__(128) unsigned char gc_tile_smem[];

// The table engine of trace_tile_kernel: DFMA sweep over a per-cell window image (see the header comment).
template <int NMAX, bool MODES>
struct TileEngine {
  static constexpr bool kStageWindow = true;
  static constexpr int kExtDoubles = 0;         // no per-thread shared scratch beyond kbuf
  static __device__ __forceinline__ int win_doubles(const FieldDev& f) { return 10 * f.tile_E; }
  static __device__ __forceinline__ const double* win_src(const FieldDev& f, int cell) {
    return f.tile_images + (size_t)cell * (10 * f.tile_E);
  }
  static __device__ __forceinline__ void rhs(const FieldDev& f, const double* win, double*, int cell, bool active,
                                             double mass, double charge, double mu, double v_ref, double inv_v_ref,
                                             double t, const double (&y)[4], double (&dy)[4]) {
    rhs_tile<NMAX, MODES>(f, win, cell, active, mass, charge, mu, v_ref, inv_v_ref, t, y, dy);
  }
};

// Body of the cell-binned persistent kernels (trace_tile_kernel, trace_mma_kernel): binning, epochs, tiles, the
// Dormand-Prince integrator of one lane per particle.  Eng supplies the window image and the right-hand side.
// mode 0: trace.  mode 1: right-hand side only (gc_rhs_eval): k1 of every particle goes to rhs_out[4][n].
// THREADS = particles per tile = threads per block; CAP = attempted steps per lane per chunk; SAMPLE = record the
// uniform-time samples of gc_trace_sampled (O9; a separate instantiation, so that gc_trace pays nothing for it).
// INTEG = 1: the symplectic explicit-implicit Euler integrator (NEXT-3) instead of Dormand-Prince: a pass of a lane is
// one field evaluation = one quasi-Newton iteration of its current step.  Lane state in the same record: y = (s, theta,
// zeta, p_zeta / (q psi0)) at the start of the step (v_par until the first pass has turned it into p_zeta), the k1 slot
// = (p_theta at the start of the step, iterate s, iterate p_zeta / (q psi0), v_par at the start of the step), n_acc =
// steps, n_rej = iterations, n_forced = iterations of the current step, `attempts` = the status the particle will
// report once its final pass has evaluated B at the reported point (v_par = q rho B / m needs it).
template <class Eng, int THREADS, int CAP, bool SAMPLE, int INTEG = 0>
__device__ __forceinline__ void trace_binned_body(const FieldDev& f, const TraceDev& p, const TileScratch& sc, int mode,
                                                  double* rhs_out) {
  cgx::grid_group grid = cgx::this_grid();
  const int tid = threadIdx.x;
  const long long gtid = (long long)blockIdx.x * THREADS + tid;
  const long long gthreads = (long long)gridDim.x * THREADS;
  const int ncell = f.ns - 3;
  const int WD = Eng::win_doubles(f);
  const int tsz = sc.tile_size;          // particles per tile (<= THREADS; smaller when the ensemble cannot fill the grid)
  constexpr double kTwoPi = 6.283185307179586476925286766559;

  double* win = reinterpret_cast<double*>(gc_tile_smem);                 // [WD] window image of the tile's cell
  double* kbuf = win + WD;                                               // [7][4][THREADS]
  double* ext = kbuf + 7 * 4 * THREADS;                                  // [Eng::kExtDoubles][THREADS] engine scratch
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(ext + Eng::kExtDoubles * THREADS);
  int* s_int = reinterpret_cast<int*>(bar + 1);                          // [0] tile id; scan space follows
  auto kb = [&](int j, int c) -> double& { return kbuf[(j * 4 + c) * THREADS + tid]; };

  if (tid == 0) mbar_init(bar, 1);
  __syncthreads();
  unsigned bar_phase = 0;

  const int chunk = (sc.chunk > 0 && sc.chunk < CAP) ? sc.chunk : CAP;
  const long long S = sc.slots;

  // Slot li takes particle i: record from the inputs, counted in its bin for the NEXT binning.
  auto init_record = [&](long long li, long long i) {
    double* r = sc.rec + li * kRecDoubles;
    double y0, y1, y2, y3, h, t = p.t0, mu = p.mu[i];
    if (mode == 1) {
      y0 = p.s0[i]; y1 = p.th0[i]; y2 = p.ze0[i]; y3 = p.vpar0[i]; h = 0.0;
    } else {
      y0 = p.s0[i]; y1 = p.th0[i]; y2 = p.ze0[i]; y3 = p.vpar0[i] * p.inv_v_ref;
      h = (p.h_inout && p.h_inout[i] > 0.0) ? p.h_inout[i] : p.h0;
      if (h < p.h_min) h = p.h_min;
    }
    const int bin = home_bin(f.ns, y0);
    int jn0 = 0;
    if constexpr (SAMPLE) {
      if (mode == 0 && p.nsamp > 0) {
        long long j = first_sample_index(p, t);
        if (j < p.nsamp && sample_time(p, j) == t) {           // a sample on t0 is the initial state
          p.samples[(0 * p.nsamp + j) * p.n + i] = y0;
          p.samples[(1 * p.nsamp + j) * p.n + i] = y1;
          p.samples[(2 * p.nsamp + j) * p.n + i] = y2;
          p.samples[(3 * p.nsamp + j) * p.n + i] = p.vpar0[i];
          ++j;
        }
        jn0 = (int)j;
      }
    }
    stcg4(r, make_double4(y0, y1, y2, y3));
    stcg4(r + 4, INTEG == 1 ? make_double4(0.0, y0, 0.0, 0.0) : make_double4(0.0, 0.0, 0.0, 0.0));
    stcg4(r + 8, make_double4(t, h, mu, __longlong_as_double(0LL)));
    __stcg(reinterpret_cast<int4*>(r + 12), make_int4(kStRunning, INTEG == 1 ? (int)kFlagFresh : 0, 0, 0));
    __stcg(reinterpret_cast<int4*>(r + 12) + 1, make_int4(0, bin, jn0, (int)i));
    atomicAdd(sc.cnt + bin, 1);
  };
  // A finished particle leaves its slot: results to the caller's arrays.
  auto flush_record = [&](long long li) {
    const double* r = sc.rec + li * kRecDoubles;
    const int4 d = __ldcg(reinterpret_cast<const int4*>(r + 12));
    const int4 g = __ldcg(reinterpret_cast<const int4*>(r + 12) + 1);
    const double4 a = ldcg4(r);
    const double4 c = ldcg4(r + 8);
    const long long i = g.w;
    if constexpr (SAMPLE) { if (p.sample_end) p.sample_end[i] = g.z; }
    p.y_out[i] = a.x;
    p.y_out[p.n + i] = a.y;
    p.y_out[2 * p.n + i] = a.z;
    p.y_out[3 * p.n + i] = a.w * p.v_ref;
    p.t_out[i] = c.x;
    p.status[i] = d.x;
    if (p.h_inout) p.h_inout[i] = c.y;
    if (p.n_acc) p.n_acc[i] = (p.resume ? p.n_acc[i] : 0) + d.z;
    if (p.n_rej) p.n_rej[i] = (p.resume ? p.n_rej[i] : 0) + d.w;
    if (p.n_forced) p.n_forced[i] = (p.resume ? p.n_forced[i] : 0) + g.x;
  };
  // Next particle to admit (GC_TRACE_RESUME: particles that finished in an earlier call are passed over), or -1.
  auto next_particle = [&]() -> long long {
    for (;;) {
      const unsigned long long i = atomicAdd(sc.next, 1ULL);
      if ((long long)i >= p.n) return -1;
      if (mode == 0 && p.resume && p.status[i] != 0) continue;
      return (long long)i;
    }
  };

  // ---- P0: the first min(slots, n) particles take the slots in order (coalesced) -----------------------------------
  if (gtid == 0) *sc.next = (unsigned long long)(S < p.n ? S : p.n);
  for (long long i = gtid; i < S; i += gthreads) {
    if (i < p.n && !(mode == 0 && p.resume && p.status[i] != 0)) {
      init_record(i, i);
    } else {                                   // nothing to trace here: the slot is refilled at the first binning
      __stcg(reinterpret_cast<int4*>(sc.rec + i * kRecDoubles + 12), make_int4(i < p.n ? kStSkip : kStEmpty, 0, 0, 0));
    }
  }
  grid.sync();

  for (;;) {
    // ---- B: segment and tile offsets (block 0) -------------------------------------------------------------------
    if (blockIdx.x == 0) {
      int* wsp = reinterpret_cast<int*>(win);                            // nbin + 2 ncell ints staged in the window space
      const int nbin = ncell * kSubBins;
      for (int b = tid; b < nbin; b += THREADS) { wsp[b] = __ldcg(sc.cnt + b); sc.cnt[b] = 0; }
      __syncthreads();
      if (tid == 0) {
        int run = 0, tiles = 0;
        for (int c = 0; c < ncell; ++c) {
          wsp[nbin + c] = run;
          wsp[nbin + ncell + c] = tiles;
          const int run0 = run;
          for (int b = c * kSubBins; b < (c + 1) * kSubBins; ++b) {      // counts become scatter cursors in place
            const int k = wsp[b];
            wsp[b] = run;
            run += k;
          }
          tiles += (run - run0 + tsz - 1) / tsz;
        }
        sc.start[ncell] = run;
        sc.tstart[ncell] = tiles;
        sc.ctrl[0] = 0; sc.ctrl[1] = 0; sc.ctrl[2] = tiles; sc.ctrl[3] = run;
        sc.ctrl[4] = (long long)__ldcg(sc.next) >= p.n;                    // every particle has been admitted
      }
      __syncthreads();
      for (int b = tid; b < nbin; b += THREADS) sc.cursor[b] = wsp[b];
      for (int c = tid; c < ncell; c += THREADS) {
        sc.start[c] = wsp[nbin + c];
        sc.tstart[c] = wsp[nbin + ncell + c];
      }
      __syncthreads();
    }
    grid.sync();
    const int ntiles = __ldcg(sc.ctrl + 2);
    if (__ldcg(sc.ctrl + 3) == 0 && __ldcg(sc.ctrl + 4) != 0) break;        // nothing runs, nothing waits

    // ---- C: scatter the running particles into cell order; slots of finished particles are flushed and handed to
    // the next unstarted particle, which joins at the next binning (it is counted in cnt now) ----------------------
    for (long long li = gtid; li < S; li += gthreads) {
      const int st_slot = __ldcg(reinterpret_cast<const int*>(sc.rec + li * kRecDoubles + 12));
      if (st_slot == kStRunning) {
        const int bin = __ldcg(reinterpret_cast<const int2*>(sc.rec + li * kRecDoubles + 14)).y;
        sc.order[atomicAdd(sc.cursor + bin, 1)] = (int)li;
      } else if (st_slot != kStEmpty) {
        if (st_slot >= 0 && mode == 0) flush_record(li);
        const long long i = next_particle();
        if (i >= 0) init_record(li, i);
        else __stcg(reinterpret_cast<int*>(sc.rec + li * kRecDoubles + 12), (int)kStEmpty);
      }
    }
    grid.sync();

    // ---- D: tiles ------------------------------------------------------------------------------------------------
    // slot of this lane in a tile: groups of 8 particles are dealt round-robin to the warps of the block, so a
    // short tile keeps every warp equally busy
    const int slot = ((((tid & 31) >> 3) * (THREADS / 32) + (tid >> 5)) << 3) | (tid & 7);
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
      const int begin = seg0 + (tile - __ldcg(sc.tstart + cell)) * tsz;
      const int count = min(tsz, seg1 - begin);
      if (Eng::kStageWindow && cell != cur_cell) {                       // stage the window: one bulk copy
        if (tid == 0) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          const unsigned bytes = (unsigned)(WD * sizeof(double));
          mbar_expect_tx(bar, bytes);
          bulk_g2s(win, Eng::win_src(f, cell), bytes, bar);
        }
        mbar_wait(bar, bar_phase);
        bar_phase ^= 1u;
        cur_cell = cell;
      }

      // lane state
      bool active = slot < count;
      long long pid = 0;
      double y[4] = {0.0, 0.0, 0.0, 0.0}, t = 0.0, h = 0.0, mu = 0.0;
      long long attempts = 0;
      int st = 0, flags = 0, n_acc = 0, n_rej = 0, n_forced = 0, jn = 0;
      int li = 0;
      if (active) {
        li = __ldcg(sc.order + begin + slot);
        const double* r = sc.rec + (long long)li * kRecDoubles;
        const double4 a = ldcg4(r);
        const double4 b = ldcg4(r + 4);
        const double4 c = ldcg4(r + 8);
        const int4 d = __ldcg(reinterpret_cast<const int4*>(r + 12));
        const int4 g = __ldcg(reinterpret_cast<const int4*>(r + 12) + 1);
        y[0] = a.x; y[1] = a.y; y[2] = a.z; y[3] = a.w;
        kb(0, 0) = b.x; kb(0, 1) = b.y; kb(0, 2) = b.z; kb(0, 3) = b.w;
        t = c.x; h = c.y; mu = c.z; attempts = __double_as_longlong(c.w);
        st = d.x; flags = d.y; n_acc = d.z; n_rej = d.w; n_forced = g.x; jn = g.z; pid = g.w;
      }
      bool running = active;                     // false once finished or parked
      bool first_chunk = true;
      bool extra = false;                        // an extra chunk: stop as soon as the epoch's first chunks are done

      for (;;) {                                 // chunks of CAP attempts
#pragma unroll 1
        for (int att = 0; att < chunk; ++att) {
          if (!__any_sync(0xffffffffu, running)) break;
          if (extra) {                           // attempts are warp-local: any warp may stop at any attempt
            int done = 0;
            if ((tid & 31) == 0) done = *reinterpret_cast<const volatile int*>(sc.ctrl + 1);
            if (__shfl_sync(0xffffffffu, done, 0) >= ntiles) break;
          }
          if constexpr (INTEG == 1) {
            // ---- one symplectic pass: the field at the current iterate (kernels_symplectic.cuh has the scheme) ------
            // k1 slot: (p_theta at the start of the step, iterate s, iterate p_zeta / (q psi0), increment of s over the
            // last step); h = increment of p_zeta / (q psi0) over the last step (the predictor of the next one)
            const double q = p.charge, unit = q * f.psi0, inv_unit = 1.0 / unit;
            const double x0 = kb(0, 1);
            double fb[4];
            Profiles pr;
            Eng::field(f, win, ext, cell, running, x0, y[1], y[2], fb, pr);
            if (running) {
              int i0c;
              double wc[4], dwc[4], chi, chi_s;
              lagrange_weights(f.ns, x0, i0c, wc, dwc);
              interp4(p.chi, 1, i0c, wc, dwc, chi, chi_s);
              const double invG = 1.0 / pr.G;
              double x1 = kb(0, 2);
              if (flags & kFlagFresh) {                        // v_par -> p_zeta = q (rho G - chi), rho = m v_par / (q B)
                x1 = (p.mass * y[3] / (q * fb[0]) * pr.G - chi) * q * inv_unit;
                flags &= ~kFlagFresh;
                if (!finite4(y[0], y[1], y[2], x1)) { st = GC_ST_NONFINITE_; running = false; }   // y[3] is still v_par
                else y[3] = x1;
              }
              const double rho = (x1 * unit / q + chi) * invG;
              if (running && (flags & kFlagFinal)) {             // the reported point: v_par = q rho B / m, then stop
                y[3] = q * rho * fb[0] / p.mass;
                st = (int)attempts;
                running = false;
              }
              if (running) {
                if (n_forced == 0) {                             // a step starts: p_theta at its start point (profiles only)
                  int i0s;
                  double ws[4], dws[4], Gs_, dG_, Is_, dI_, chis_, dchis_;
                  lagrange_weights(f.ns, y[0], i0s, ws, dws);
                  interp4(f.G, 1, i0s, ws, dws, Gs_, dG_);
                  interp4(f.I, 1, i0s, ws, dws, Is_, dI_);
                  interp4(p.chi, 1, i0s, ws, dws, chis_, dchis_);
                  kb(0, 0) = q * fma((y[3] * unit / q + chis_) / Gs_, Is_, f.psi0 * y[0]);
                }
                const double rho_s = (chi_s - rho * pr.Gs) * invG;
                const double pth = q * fma(rho, pr.I, f.psi0 * x0);
                const double D = q * (f.psi0 + rho_s * pr.I + rho * pr.Is);
                const double dpth_dpz = pr.I * invG;
                const double qr = q * rho;
                const double dHdB = fma(qr * qr / p.mass, fb[0], mu);
                const double F1 = pth - kb(0, 0) + p.sym_dt * dHdB * fb[2];
                const double F2 = (x1 - y[3]) * unit + p.sym_dt * dHdB * fb[3];
                const double dpz = -F2;
                const double ds = -(F1 + dpth_dpz * dpz) / D;
                const double dx1 = dpz * inv_unit;
                ++n_forced;
                ++n_rej;
                bool failed = !isfinite(ds) || !isfinite(dx1);
                if (!failed) {
                  const double xn0 = x0 + ds, xn1 = x1 + dx1;
                  kb(0, 1) = xn0; kb(0, 2) = xn1;
                  if (fabs(ds) <= p.sym_tol * fmax(1.0, fabs(xn0)) && fabs(dx1) <= p.sym_tol * fmax(1.0, fabs(xn1))) {
                    const double H_s = qr * q * rho_s * fb[0] * fb[0] / p.mass + dHdB * fb[1];
                    const double H_pz = qr * fb[0] * fb[0] / (p.mass * pr.G);
                    const double th_new = fma(p.sym_dt, H_s / D, y[1]);
                    const double ze_new = fma(p.sym_dt, H_pz - H_s * dpth_dpz / D, y[2]);
                    if (!finite4(xn0, th_new, ze_new, xn1)) {
                      failed = true;
                    } else {
                      kb(0, 3) = xn0 - y[0];                     // the predictor of the next step
                      h = xn1 - y[3];
                      y[0] = xn0; y[1] = th_new; y[2] = ze_new; y[3] = xn1;
                      n_forced = 0;
                      ++n_acc;
                      t = __dadd_rn(p.t0, __dmul_rn((double)n_acc, p.sym_dt));
                      int stop = -1;
                      if (y[0] >= p.s_loss) stop = 1;
                      else if (y[0] <= p.s_min) stop = 2;
                      else if ((long long)n_acc >= p.sym_nsteps) stop = 0;
                      if (stop >= 0) {
                        flags |= kFlagFinal; attempts = stop;     // next pass: B at the end point
                      } else {
                        kb(0, 1) = y[0] + kb(0, 3);              // start the next step from the extrapolation
                        kb(0, 2) = y[3] + h;
                      }
                      const int hc = home_cell(f.ns, y[0]);
                      if (hc < cell - 1 || hc > cell + 1) running = false;   // parked until the next binning
                    }
                  } else if (n_forced >= p.sym_max_iter) {
                    failed = true;
                  }
                }
                if (failed) {                                    // report the state before the failed step: one more
                  flags |= kFlagFinal; attempts = GC_ST_NONFINITE_;   // pass at that point for its v_par
                  kb(0, 1) = y[0]; kb(0, 2) = y[3];
                  n_forced = 0;
                }
              }
            }
            continue;
          }
          // stage 0 gives k1 to lanes that do not carry one yet (first epoch; gc_rhs_eval)
          const bool do_k1 = __any_sync(0xffffffffu, running && !(flags & kFlagHaveK1));
          double h_try = h, yn[4] = {y[0], y[1], y[2], y[3]};
          bool clipped = false;
          const bool forced = (flags & kFlagPrevRejected) && p.h_min > 0.0 && h == p.h_min;
          if (mode == 0 && running && t < p.t_max) {
            if (t + h_try >= p.t_max) { h_try = p.t_max - t; clipped = true; }
            if (!(t + h_try > t)) { st = GC_ST_NONFINITE_; running = false; }       // step underflow
          }
#pragma unroll 1
          for (int stage = do_k1 ? 0 : 1; stage <= 6; ++stage) {
            if (stage > 0 && !__any_sync(0xffffffffu, running)) break;
            double ys[4], ts;
            if (stage == 0) {
              ys[0] = y[0]; ys[1] = y[1]; ys[2] = y[2]; ys[3] = y[3];
              ts = t;
            } else {
              double acc[4] = {0.0, 0.0, 0.0, 0.0};
              for (int j = 0; j < stage; ++j) {
                const double a = cDpA[stage][j];
#pragma unroll
                for (int c = 0; c < 4; ++c) acc[c] = fma(a, kb(j, c), acc[c]);
              }
#pragma unroll
              for (int c = 0; c < 4; ++c) ys[c] = fma(h_try, acc[c], y[c]);
              ts = fma(cDpC[stage], h_try, t);
              if (stage == 6) { yn[0] = ys[0]; yn[1] = ys[1]; yn[2] = ys[2]; yn[3] = ys[3]; }
            }
            double dy[4] = {0.0, 0.0, 0.0, 0.0};
            const bool lane_on = running && (stage > 0 || !(flags & kFlagHaveK1));
            Eng::rhs(f, win, ext, cell, lane_on, p.mass, p.charge, mu, p.v_ref, p.inv_v_ref, ts, ys, dy);
            if (lane_on) {
              kb(stage, 0) = dy[0]; kb(stage, 1) = dy[1]; kb(stage, 2) = dy[2]; kb(stage, 3) = dy[3];
              if (stage == 0) {
                flags |= kFlagHaveK1;
                if (mode == 1) {
#pragma unroll
                  for (int c = 0; c < 4; ++c) rhs_out[(long long)c * p.n + pid] = dy[c];
                  st = 0; running = false;
                } else if (!finite4(y[0], y[1], y[2], y[3]) || !finite4(dy[0], dy[1], dy[2], dy[3])) {
                  st = GC_ST_NONFINITE_; running = false;
                } else if (!(t < p.t_max)) {
                  st = 0; running = false;
                }
              }
            }
          }
          if (running) {
            ++attempts;
            double accn = 0.0;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
              double e = 0.0;
              for (int j = 0; j < 7; ++j) e = fma(cDpE[j], kb(j, c), e);
              const double delta = h_try * e;
              const double sk = fma(p.rtol, fmax(fabs(y[c]), fabs(yn[c])), p.atol);
              const double r = delta / sk;
              accn = fma(r, r, accn);
            }
            const double err = sqrt(accn * 0.25);
            const bool finite = finite4(yn[0], yn[1], yn[2], yn[3]) &&
                                finite4(kb(6, 0), kb(6, 1), kb(6, 2), kb(6, 3)) && isfinite(err);
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
              bool zeta_section = true;
              if constexpr (SAMPLE) {                                     // O8b lives in the diagnostics build only
                if (p.section == 1) {
                  zeta_section = false;
                  if (p.poincare_capacity > 0 && bounce_crossed(y[3], yn[3])) {
                    double hk1[4], hk7[4], hd[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                      double dd = 0.0;
                      for (int j = 0; j < 7; ++j) dd = fma(cDpD[j], kb(j, c), dd);
                      hk1[c] = h_try * kb(0, c); hk7[c] = h_try * kb(6, c); hd[c] = h_try * dd;
                    }
                    bounce_emit(y, yn, hk1, hk7, hd, pid, t, h_try, p.poincare, p.poincare_capacity, p.poincare_count);
                  }
                }
              }
              if (zeta_section && p.poincare_capacity > 0 && floor(y[2] / kTwoPi) != floor(yn[2] / kTwoPi)) {
                Dense3 d;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                  double dd = 0.0;
                  for (int j = 0; j < 7; ++j) dd = fma(cDpD[j], kb(j, c), dd);
                  d.r1[c] = y[c];
                  d.r2[c] = yn[c] - y[c];
                  d.r3[c] = h_try * kb(0, c) - d.r2[c];
                  d.r4[c] = d.r2[c] - h_try * kb(6, c) - d.r3[c];
                  d.r5[c] = h_try * dd;
                }
                poincare_emit(d, pid, t, h_try, y[2], yn[2], p.poincare, p.poincare_capacity, p.poincare_count);
              }
              const double t_new = clipped ? p.t_max : t + h_try;
              if constexpr (SAMPLE) {                                     // O9
                if (jn < p.nsamp && sample_time(p, jn) <= t_new) {
                  double hd[4];
#pragma unroll
                  for (int c = 0; c < 4; ++c) {
                    double dd = 0.0;
                    for (int j = 0; j < 7; ++j) dd = fma(cDpD[j], kb(j, c), dd);
                    hd[c] = h_try * dd;
                  }
                  while (jn < p.nsamp) {
                    const double tj = sample_time(p, jn);
                    if (tj > t_new) break;
                    const double tau = (tj - t) / h_try;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                      const double v = dense_component(y[c], yn[c], h_try * kb(0, c), h_try * kb(6, c), hd[c], tau);
                      p.samples[((long long)c * p.nsamp + jn) * p.n + pid] = c == 3 ? v * p.v_ref : v;
                    }
                    ++jn;
                  }
                }
              }
              const bool lost_now = yn[0] >= p.s_loss;
              if constexpr (SAMPLE) {                                     // O7b lives in the diagnostics build only
                if (lost_now && p.refine_loss && y[0] < p.s_loss) {
                  double hd[4];
#pragma unroll
                  for (int c = 0; c < 4; ++c) {
                    double dd = 0.0;
                    for (int j = 0; j < 7; ++j) dd = fma(cDpD[j], kb(j, c), dd);
                    hd[c] = h_try * dd;
                  }
                  const double tau = loss_root(y[0], yn[0], h_try * kb(0, 0), h_try * kb(6, 0), hd[0], p.s_loss);
#pragma unroll
                  for (int c = 0; c < 4; ++c)
                    yn[c] = dense_component(y[c], yn[c], h_try * kb(0, c), h_try * kb(6, c), hd[c], tau);
                  t = fma(tau, h_try, t);
                } else {
                  t = t_new;
                }
              } else {
                t = t_new;
              }
#pragma unroll
              for (int c = 0; c < 4; ++c) { y[c] = yn[c]; kb(0, c) = kb(6, c); }
              ++n_acc;
              if (forced) ++n_forced;
              flags &= ~kFlagPrevRejected;
              if (!clipped) h = h_next;
              if (h < p.h_min) h = p.h_min;
              if (lost_now) st = 1;
              else if (y[0] <= p.s_min) st = 2;
              else if (clipped) st = 0;
              else if (attempts >= p.max_steps) st = 3;
              if (st != kStRunning) running = false;
              else {
                const int hc = home_cell(f.ns, y[0]);
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
          if (next >= ntiles && nrun * 2 >= tsz) {
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
        double* r = sc.rec + (long long)li * kRecDoubles;
        const int hb = home_bin(f.ns, y[0]);
        stcg4(r, make_double4(y[0], y[1], y[2], y[3]));
        stcg4(r + 4, make_double4(kb(0, 0), kb(0, 1), kb(0, 2), kb(0, 3)));
        stcg4(r + 8, make_double4(t, h, mu, __longlong_as_double(attempts)));
        __stcg(reinterpret_cast<int4*>(r + 12), make_int4(st, flags, n_acc, n_rej));
        __stcg(reinterpret_cast<int4*>(r + 12) + 1, make_int4(n_forced, hb, jn, (int)pid));
        if (st == kStRunning) atomicAdd(sc.cnt + hb, 1);
      }
      __syncthreads();                                                   // window / kbuf / s_int are reused
    }
    grid.sync();
  }

  // ---- the particles still in the slots -----------------------------------------------------------------------------
  if (mode == 0) {
    for (long long li = gtid; li < S; li += gthreads)
      if (__ldcg(reinterpret_cast<const int*>(sc.rec + li * kRecDoubles + 12)) >= 0) flush_record(li);
  }
}

template <int NMAX, bool MODES, bool SAMPLE>
__global__ void __launch_bounds__(kTileThreads, 2)
trace_tile_kernel(FieldDev f, TraceDev p, TileScratch sc, int mode, double* rhs_out) {
  trace_binned_body<TileEngine<NMAX, MODES>, kTileThreads, kTileCap, SAMPLE>(f, p, sc, mode, rhs_out);
}

}  // namespace gc
