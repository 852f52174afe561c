// gcorbit_api.cu -- C ABI of libgcorbit.so (include/gcorbit.h): table upload and packing, kernel dispatch.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -shared -Xcompiler -fPIC
#include "../../include/gcorbit.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

namespace gc { constexpr int GC_ST_NONFINITE_ = 4; }
#include "kernels_generic.cuh"
#include "kernels_lane.cuh"
#include "kernels_symplectic.cuh"
#include "kernels_warp.cuh"
#include "kernels_tile.cuh"
#include "kernels_mma.cuh"

namespace {

thread_local std::string g_last_error;

int fail(int code, const std::string& msg) {
  g_last_error = msg;
  return code;
}

#define GC_CUDA(expr)                                                                          \
  do {                                                                                         \
    cudaError_t e_ = (expr);                                                                   \
    if (e_ != cudaSuccess)                                                                     \
      return fail(e_ == cudaErrorMemoryAllocation ? GC_ENOMEM : GC_ECUDA,                      \
                  std::string(#expr) + ": " + cudaGetErrorString(e_));                         \
  } while (0)

template <typename T>
int upload(const T* host, size_t count, T** dev) {
  *dev = nullptr;
  if (count == 0) return GC_OK;
  GC_CUDA(cudaMalloc((void**)dev, count * sizeof(T)));
  GC_CUDA(cudaMemcpy(*dev, host, count * sizeof(T), cudaMemcpyHostToDevice));
  return GC_OK;
}

bool all_finite(const double* p, size_t n) {
  for (size_t i = 0; i < n; ++i)
    if (!std::isfinite(p[i])) return false;
  return true;
}

}  // namespace

struct gc_field {
  gc::FieldDev dev{};
  std::vector<void*> allocs;
  int kernel = GC_KERNEL_AUTO;      // requested choice; resolved per call by resolve_kernel()
  bool warp_ok = false;
  bool tile_ok = false;
  int nit_main_inst = 0;            // instantiated (padded) main iteration count
  int sm_count = 0;
  int tile_smem = 0;                // dynamic shared memory of the tile kernel
  int tile_blocks_per_sm = 0;       // co-resident blocks per SM (cooperative launch)
  // workspace of gc_trace_host, kept between calls (cudaMalloc / cudaFree per call cost up to 200 ms now and then)
  cudaStream_t host_stream = nullptr;
  void* host_slab = nullptr;
  size_t host_slab_bytes = 0;
  // per-call scratch of the trace kernels comes from a pool of the field that keeps what it is given back (the
  // default pool of the device returns freed memory to the driver at every synchronisation, so a caller that
  // synchronises after each call -- gc_trace_host does -- paid a fresh 13..128 MB allocation per call)
  cudaMemPool_t pool = nullptr;
  long long wave_particles = 0;     // GC_OPT_WAVE_PARTICLES (0 = automatic)
  int chunk_attempts = 0;           // GC_OPT_CHUNK_ATTEMPTS (0 = the kernel's default)
  std::atomic<bool> host_busy{false};   // gc_trace_host is not re-entrant on one field: overlapping calls get GC_EINVAL
  bool mma_ok = false;
  bool extra = false;               // NEXT-4 tables present (bmns, kmnc or kmns): mma or generic kernel only
  int mma_smem = 0;                 // dynamic shared memory of the mma kernel
  int mma_blocks_per_sm = 0;
  double* grid = nullptr;           // NEXT-2: node values of the 3-D interpolant (gc_field_set_grid), else nullptr
};

namespace {

// ---- warp-kernel instantiations -------------------------------------------------------------------------------
// NIT_MAIN is padded up to the next compiled size; NX in {1, 2}; NREG = iterations kept in registers.
struct WarpInst {
  int nit_main, nx;
  bool modes;
  const void* trace_fn;
  const void* rhs_fn;
  int smem_bytes;
};

template <int NIT_MAIN, int NX, bool MODES, int NREG>
WarpInst make_inst() {
  constexpr int NSM = NIT_MAIN + NX - NREG;
  return WarpInst{NIT_MAIN, NX, MODES,
                  (const void*)gc::trace_warp_kernel<NIT_MAIN, NX, MODES, NREG>,
                  (const void*)gc::rhs_eval_warp_kernel<NIT_MAIN, NX, MODES, NREG>,
                  (int)(sizeof(gc::WarpScratch) * gc::kWarpsPerBlock +
                        (size_t)gc::kWarpsPerBlock * NSM * 4 * 32 * sizeof(double))};
}

#ifndef GC_NREG_LARGE
#define GC_NREG_LARGE 18
#endif

const std::vector<WarpInst>& warp_instances() {
  static const std::vector<WarpInst> v = {
      make_inst<5, 1, false, 6>(),  make_inst<5, 1, true, 6>(),  make_inst<5, 2, true, 7>(),
      make_inst<9, 1, false, 10>(), make_inst<9, 1, true, 10>(), make_inst<9, 2, true, 11>(),
      make_inst<17, 1, false, (GC_NREG_LARGE < 18 ? GC_NREG_LARGE : 18)>(),
      make_inst<17, 1, true, (GC_NREG_LARGE < 18 ? GC_NREG_LARGE : 18)>(),
      make_inst<17, 2, true, (GC_NREG_LARGE < 19 ? GC_NREG_LARGE : 19)>(),
  };
  return v;
}

const WarpInst* find_inst(const gc_field* f) {
  if (!f->warp_ok) return nullptr;
  for (const WarpInst& w : warp_instances())
    if (w.nit_main == f->nit_main_inst && w.nx == f->dev.nx && w.modes == (f->dev.nk > 0)) return &w;
  return nullptr;
}

int ensure_smem(const void* fn, int bytes) {
  GC_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  return GC_OK;
}

// Dynamic shared memory the binned kernels may ask for: two blocks per SM must fit.  The attribute belongs to the
// kernel FUNCTION, not to a field (two live fields can share an instantiation with different window sizes), so every
// instantiation is raised to this one cap and never lowered.
constexpr int kBinnedSmemCap = 110 * 1024;

// Record slots of the binned kernels when the caller does not say (GC_OPT_WAVE_PARTICLES): 2^18 records of 128 B =
// 32 MB, a quarter of the 126 MB L2.
constexpr long long kAutoWaveParticles = 1 << 18;

// Packed rows[node][it][lane] of the warp kernel (kernels_warp.cuh header comment).
int pack_rows(gc_field* f, const gc_field_desc* d) {
  gc::FieldDev& v = f->dev;
  const int M = v.M, N = v.N;
  f->warp_ok = false;
  if (N > gc::kMaxN || M > 28 || f->extra) return GC_OK;
  int cl_log = 5;
  if (N > 0) {
    cl_log = 1;
    while ((1 << cl_log) < 2 * N) ++cl_log;
  }
  const int groups = 32 >> cl_log;
  const int nit_main = N > 0 ? (M + 1 + groups - 1) / groups : 0;
  const int nx = (M + 4 + d->nk + 31) / 32;
  int inst = -1;
  for (const WarpInst& w : warp_instances())
    if (w.nit_main >= nit_main && w.nit_main * groups <= gc::kMaxRowsM && w.nx == nx &&
        w.modes == (d->nk > 0) && (inst < 0 || w.nit_main < inst))
      inst = w.nit_main;
  if (inst < 0) return GC_OK;
  const int nit = inst + nx;
  std::vector<double> rows((size_t)d->ns * nit * 32, 0.0);
  const int cl = 1 << cl_log;
  for (int node = 0; node < d->ns; ++node) {
    double* row = rows.data() + (size_t)node * nit * 32;
    for (int k = 0; k < d->nh; ++k) {
      const int m = d->xm[k], n = d->xn[k];
      const double b = d->bmnc[(size_t)node * d->nh + k];
      if (n == 0) {
        row[(size_t)inst * 32 + m] += b;                      // n = 0 column: extra index m
        continue;
      }
      const int an = n > 0 ? n : -n;
      const int g = m % groups, it = m / groups;
      const int laneP = g * cl + 2 * (an - 1), laneQ = laneP + 1;
      row[(size_t)it * 32 + laneP] += b;                      // P = b(m,n) + b(m,-n)
      row[(size_t)it * 32 + laneQ] += n > 0 ? b : -b;         // Q = b(m,n) - b(m,-n)
    }
    auto extra = [&](int e) -> double& { return row[(size_t)(inst + e / 32) * 32 + (e % 32)]; };
    extra(M + 1) = d->G[node];
    extra(M + 2) = d->I[node];
    extra(M + 3) = d->iota[node];
    for (int k = 0; k < d->nk; ++k) extra(M + 4 + k) = d->phihat[(size_t)node * d->nk + k];
  }
  double* dev_rows = nullptr;
  int rc = upload(rows.data(), rows.size(), &dev_rows);
  if (rc != GC_OK) return rc;
  f->allocs.push_back(dev_rows);
  v.rows = dev_rows;
  v.cl_log = cl_log;
  v.nit_main = inst;
  v.nx = nx;
  v.nit = nit;
  f->nit_main_inst = inst;
  f->warp_ok = true;
  return GC_OK;
}

// ---- tile-kernel instantiations and window images -------------------------------------------------------------
template <bool SAMPLE>
const void* tile_fn_t(const gc_field* f) {
  const bool modes = f->dev.nk > 0;
  if (f->dev.tile_nmax == 8)
    return modes ? (const void*)gc::trace_tile_kernel<8, true, SAMPLE> : (const void*)gc::trace_tile_kernel<8, false, SAMPLE>;
  return modes ? (const void*)gc::trace_tile_kernel<16, true, SAMPLE> : (const void*)gc::trace_tile_kernel<16, false, SAMPLE>;
}
const void* tile_fn(const gc_field* f, bool sample = false) { return sample ? tile_fn_t<true>(f) : tile_fn_t<false>(f); }

template <bool SAMPLE>
const void* mma_fn_t(const gc_field* f) {
  const bool modes = f->dev.nk > 0;
  if (f->extra)                                            // NEXT-4 tables: the 16/16 layout with the extra sweeps
    return modes ? (const void*)gc::trace_mma_kernel<2, 4, true, SAMPLE, true> : (const void*)gc::trace_mma_kernel<2, 4, false, SAMPLE, true>;
  if (f->dev.mma_MT == 1)
    return modes ? (const void*)gc::trace_mma_kernel<1, 2, true, SAMPLE> : (const void*)gc::trace_mma_kernel<1, 2, false, SAMPLE>;
  return modes ? (const void*)gc::trace_mma_kernel<2, 4, true, SAMPLE> : (const void*)gc::trace_mma_kernel<2, 4, false, SAMPLE>;
}
const void* mma_fn(const gc_field* f, bool sample = false) { return sample ? mma_fn_t<true>(f) : mma_fn_t<false>(f); }
// the symplectic integrator on the mma engine (static fields without NEXT-4 tables)
const void* mma_sym_fn(const gc_field* f) {
  return f->dev.mma_MT == 1 ? (const void*)gc::trace_mma_symplectic_kernel<1, 2>
                            : (const void*)gc::trace_mma_symplectic_kernel<2, 4>;
}

int resolve_kernel(const gc_field* f, int64_t n) {
  if (f->dev.grid) return GC_KERNEL_GRID;                  // the field IS the interpolant while a grid is set
  if (f->kernel != GC_KERNEL_AUTO) return f->kernel;
  // switch-over measured on B200 (profiles/r2_ensemble_size_sweep.md): the warp kernel wins below it
  const int64_t nmin = (f->dev.M <= 8 && f->dev.N <= 8) ? GC_TILE_MIN_PARTICLES_SMALL : GC_TILE_MIN_PARTICLES;
  if (f->mma_ok && n >= nmin) return GC_KERNEL_MMA;
  if (f->tile_ok && n >= nmin) return GC_KERNEL_TILE;
  return f->warp_ok ? GC_KERNEL_WARP : GC_KERNEL_GENERIC;
}

// images[cell][10 E]: [E][6] node rows cell-1 .. cell+4 (zero where the row does not exist), then [E][4] rows
// cell .. cell+3 (kernels_tile.cuh).  Entries: per m, b(m,0) then (P, Q)(m,n) for n = 1..NMAX with
// P = b(m,n) + b(m,-n), Q = b(m,n) - b(m,-n); then G, I, iota; then the nk mode amplitudes.
int pack_tile_images(gc_field* f, const gc_field_desc* d) {
  gc::FieldDev& v = f->dev;
  f->tile_ok = false;
  if (v.N > 16 || f->extra) return GC_OK;
  const int nmax = v.N <= 8 ? 8 : 16;
  const int rowlen = 1 + 2 * nmax;
  const int E = (v.M + 1) * rowlen + 3 + d->nk;
  const int smem = (int)((size_t)10 * E * sizeof(double) + (size_t)7 * 4 * gc::kTileThreads * sizeof(double) + 64);
  if (smem > kBinnedSmemCap) return GC_OK;                 // two blocks per SM must fit
  const int ncell = d->ns - 3;
  if ((size_t)(gc::kSubBins + 2) * ncell * sizeof(int) > (size_t)10 * E * sizeof(double)) return GC_OK;   // scan space (phase B)
  // node-major entry rows first
  std::vector<double> rows((size_t)d->ns * E, 0.0);
  for (int node = 0; node < d->ns; ++node) {
    double* row = rows.data() + (size_t)node * E;
    for (int k = 0; k < d->nh; ++k) {
      const int m = d->xm[k], n = d->xn[k];
      const double b = d->bmnc[(size_t)node * d->nh + k];
      double* r = row + (size_t)m * rowlen;
      if (n == 0) { r[0] += b; continue; }
      const int an = n > 0 ? n : -n;
      r[2 * an - 1] += b;                                  // P
      r[2 * an] += n > 0 ? b : -b;                         // Q
    }
    double* x = row + (size_t)(v.M + 1) * rowlen;
    x[0] = d->G[node]; x[1] = d->I[node]; x[2] = d->iota[node];
    for (int k = 0; k < d->nk; ++k) x[3 + k] = d->phihat[(size_t)node * d->nk + k];
  }
  std::vector<double> img((size_t)ncell * 10 * E, 0.0);
  for (int c = 0; c < ncell; ++c) {
    double* A = img.data() + (size_t)c * 10 * E;
    double* Bq = A + (size_t)6 * E;
    for (int e = 0; e < E; ++e) {
      for (int j = 0; j < 6; ++j) {
        const int node = c - 1 + j;
        if (node >= 0 && node < d->ns) A[(size_t)e * 6 + j] = rows[(size_t)node * E + e];
      }
      for (int j = 0; j < 4; ++j) Bq[(size_t)e * 4 + j] = rows[(size_t)(c + j) * E + e];
    }
  }
  double* dev_img = nullptr;
  int rc = upload(img.data(), img.size(), &dev_img);
  if (rc != GC_OK) return rc;
  f->allocs.push_back(dev_img);
  v.tile_images = dev_img;
  v.tile_E = E;
  v.tile_nmax = nmax;
  f->tile_smem = smem;
  const void* fn = tile_fn(f);
  GC_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, kBinnedSmemCap));
  GC_CUDA(cudaFuncSetAttribute(tile_fn(f, true), cudaFuncAttributeMaxDynamicSharedMemorySize, kBinnedSmemCap));
  int per_sm = 0, per_sm_diag = 0;
  GC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, gc::kTileThreads, (size_t)smem));
  GC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_diag, tile_fn(f, true), gc::kTileThreads, (size_t)smem));
  if (per_sm_diag < per_sm) per_sm = per_sm_diag;
  if (per_sm < 1) return GC_OK;
  int coop = 0, devid = 0;
  GC_CUDA(cudaGetDevice(&devid));
  GC_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, devid));
  if (!coop) return GC_OK;
  f->tile_blocks_per_sm = per_sm;
  f->tile_ok = true;
  return GC_OK;
}

// image[ns + 4][RS] of the mma kernel (kernels_mma.cuh): image row = node + 2; per row the DMMA B fragments
// (P, Q)(m, n) in lane order, then b(m, 0), b(0, n), G, I, iota and the mode amplitudes.
// `tab` = bmnc (with profiles and modes) or one of the NEXT-4 tables (series coefficients only; sin_table: the
// entries multiply sin(m th - n nfp ze), so b(0, -n) enters the m = 0 row with the opposite sign).
template <int MT, int KS>
void fill_mma_rows(const gc_field_desc* d, int RS, std::vector<double>& img, const double* tab = nullptr,
                   bool sin_table = false) {
  using R = gc::MmaRow<MT, KS>;
  const bool main_table = tab == nullptr;
  if (main_table) tab = d->bmnc;
  for (int node = 0; node < d->ns; ++node) {
    double* row = img.data() + (size_t)(node + 2) * RS;
    for (int k = 0; k < d->nh; ++k) {
      const int m = d->xm[k], n = d->xn[k];
      const double b = tab[(size_t)node * d->nh + k];
      const int an = n > 0 ? n : -n;
      if (m == 0) { row[R::kM0 + an] += (sin_table && n < 0) ? -b : b; continue; }
      if (n == 0) { row[R::kN0 + m - 1] += b; continue; }
      const int T = (m - 1) / 8, g = (m - 1) % 8, j = (an - 1) / 4, q = (an - 1) % 4;
      double* e = row + R::kFrag + ((size_t)(T * KS + j) * 32 + 4 * g + q) * 2;
      e[0] += b;                                           // P = b(m,n) + b(m,-n)
      e[1] += n > 0 ? b : -b;                              // Q = b(m,n) - b(m,-n)
    }
    if (!main_table) continue;
    row[R::kProf] = d->G[node]; row[R::kProf + 1] = d->I[node]; row[R::kProf + 2] = d->iota[node];
    for (int k = 0; k < d->nk; ++k) row[R::kModes + k] = d->phihat[(size_t)node * d->nk + k];
  }
}

int pack_mma_image(gc_field* f, const gc_field_desc* d) {
  gc::FieldDev& v = f->dev;
  f->mma_ok = false;
  if (v.N > 16 || v.M > 16) return GC_OK;
  const bool small = v.M <= 8 && v.N <= 8 && !f->extra;
  const int MT = small ? 1 : 2, KS = small ? 2 : 4;
  const int RS = small ? gc::MmaRow<1, 2>::stride(d->nk) : gc::MmaRow<2, 4>::stride(d->nk);
  const int smem = (int)((size_t)gc::kMmaWinRows * RS * sizeof(double) + (size_t)(7 * 4 + 2 * gc::kMmaWtab) * gc::kMmaThreads * sizeof(double) + 64);
  if (smem > kBinnedSmemCap) return GC_OK;
  const int ncell = d->ns - 3;
  if ((size_t)(gc::kSubBins + 2) * ncell * sizeof(int) > (size_t)gc::kMmaWinRows * RS * sizeof(double)) return GC_OK;
  std::vector<double> img((size_t)(d->ns + 4) * RS, 0.0);
  if (small) fill_mma_rows<1, 2>(d, RS, img); else fill_mma_rows<2, 4>(d, RS, img);
  double* dev_img = nullptr;
  int rc = upload(img.data(), img.size(), &dev_img);
  if (rc != GC_OK) return rc;
  f->allocs.push_back(dev_img);
  v.mma_image = dev_img;
  v.mma_RS = RS; v.mma_MT = MT; v.mma_KS = KS;
  const double* extra_tab[3] = {d->bmns, d->kmnc, d->kmns};
  const double** extra_dst[3] = {&v.mma_image_bs, &v.mma_image_kc, &v.mma_image_ks};
  for (int x = 0; x < 3; ++x) {
    if (!extra_tab[x]) continue;
    std::vector<double> ximg((size_t)(d->ns + 4) * RS, 0.0);
    fill_mma_rows<2, 4>(d, RS, ximg, extra_tab[x], x != 1);
    double* dev_x = nullptr;
    rc = upload(ximg.data(), ximg.size(), &dev_x);
    if (rc != GC_OK) return rc;
    f->allocs.push_back(dev_x);
    *extra_dst[x] = dev_x;
  }
  f->mma_smem = smem;
  const void* fn = mma_fn(f);
  GC_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, kBinnedSmemCap));
  GC_CUDA(cudaFuncSetAttribute(mma_fn(f, true), cudaFuncAttributeMaxDynamicSharedMemorySize, kBinnedSmemCap));
  if (!f->extra) GC_CUDA(cudaFuncSetAttribute(mma_sym_fn(f), cudaFuncAttributeMaxDynamicSharedMemorySize, kBinnedSmemCap));
  int per_sm = 0, per_sm_diag = 0;                         // the plain and the diagnostics build share one grid size
  GC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, gc::kMmaThreads, (size_t)smem));
  GC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_diag, mma_fn(f, true), gc::kMmaThreads, (size_t)smem));
  if (per_sm_diag < per_sm) per_sm = per_sm_diag;
  if (per_sm < 1) return GC_OK;
  int coop = 0, devid = 0;
  GC_CUDA(cudaGetDevice(&devid));
  GC_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, devid));
  if (!coop) return GC_OK;
  f->mma_blocks_per_sm = per_sm;
  f->mma_ok = true;
  return GC_OK;
}

// Blocks and particles per tile for n particles: full tiles when the ensemble fills the persistent grid, else
// tiles shrunk (to a multiple of 8 = one DMMA group; smaller tiles were measured and gain nothing) so that every
// block gets one.
long long tile_geometry(const gc_field* f, long long n, bool mma, int* tile_size) {
  const int threads = mma ? gc::kMmaThreads : gc::kTileThreads;
  const long long grid = (long long)f->sm_count * (mma ? f->mma_blocks_per_sm : f->tile_blocks_per_sm);
  long long tsz = threads;
  if (n < grid * threads) {
    tsz = ((n + grid - 1) / grid + 7) / 8 * 8;
    if (tsz < 8) tsz = 8;
    if (tsz > threads) tsz = threads;
  }
  long long blocks = (n + tsz - 1) / tsz;
  if (blocks > grid) blocks = grid;
  if (blocks < 1) blocks = 1;
  *tile_size = (int)tsz;
  return blocks;
}

// Record slots of the binned kernels: the 128-byte records must stay in L2 between epochs, so a large ensemble
// streams through a fixed number of slots (kernels_tile.cuh).
long long wave_size(const gc_field* f, long long n) {
  const long long slots = f->wave_particles > 0 ? f->wave_particles : kAutoWaveParticles;
  if (n <= slots + slots / 4) return n > 0 ? n : 1;        // every particle has its own slot
  return slots;
}

// One cooperative launch of the tile or mma kernel (mode 0 trace, mode 1 right-hand side only) with its scratch.
int launch_tile(const gc_field* f, gc::TraceDev& t, int mode, double* rhs_out, cudaStream_t st, bool mma = false,
                bool symplectic = false) {
  const int ncell = f->dev.ns - 3;
  const size_t n = (size_t)t.n;
  const long long wave = wave_size(f, (long long)n);
  const size_t wn = (size_t)wave;
  const size_t rec_bytes = wn * gc::kRecDoubles * sizeof(double);
  const size_t nbin = (size_t)ncell * gc::kSubBins;
  const size_t int_count = ((wn + 1) & ~(size_t)1) + 2 * nbin + (size_t)2 * (ncell + 1) + 8 + 4;
  unsigned char* slab = nullptr;
  GC_CUDA(cudaMallocFromPoolAsync((void**)&slab, rec_bytes + int_count * sizeof(int), f->pool, st));
  gc::TileScratch sc{};
  sc.slots = wave;
  sc.chunk = f->chunk_attempts;
  sc.rec = reinterpret_cast<double*>(slab);
  int* ip = reinterpret_cast<int*>(slab + rec_bytes);
  sc.order = ip; ip += (wn + 1) & ~(size_t)1;
  sc.cnt = ip; ip += nbin;
  sc.cursor = ip; ip += nbin;
  sc.start = ip; ip += ncell + 1;
  sc.tstart = ip; ip += ncell + 1;
  sc.ctrl = ip; ip += 8;
  ip += ((reinterpret_cast<uintptr_t>(ip) & 7) ? 1 : 0);   // the 64-bit input cursor
  sc.next = reinterpret_cast<unsigned long long*>(ip);
  GC_CUDA(cudaMemsetAsync(sc.cnt, 0, (2 * nbin + (size_t)2 * (ncell + 1) + 8 + 4) * sizeof(int), st));
  int per_tile = 0;
  long long blocks = tile_geometry(f, (long long)wn, mma, &per_tile);
  sc.tile_size = per_tile;
  gc::FieldDev fd = f->dev;
  void* args[] = {(void*)&fd, (void*)&t, (void*)&sc, (void*)&mode, (void*)&rhs_out};
  const bool sample = mode == 0 && (t.nsamp > 0 || t.section != 0 || t.refine_loss != 0);   // the diagnostics build of the kernel
  const cudaError_t le =
      mma ? cudaLaunchCooperativeKernel(symplectic ? mma_sym_fn(f) : mma_fn(f, sample), dim3((unsigned)blocks),
                                        dim3(gc::kMmaThreads), args, (size_t)f->mma_smem, st)
          : cudaLaunchCooperativeKernel(tile_fn(f, sample), dim3((unsigned)blocks), dim3(gc::kTileThreads), args,
                                        (size_t)f->tile_smem, st);
  const cudaError_t fe = cudaFreeAsync(slab, st);           // also on a failed launch: the scratch must not leak
  GC_CUDA(le);
  GC_CUDA(fe);
  return GC_OK;
}

// One launch of the lane kernel (generic field or 3-D interpolant): persistent grid, atomic particle queue.
const void* lane_fn(int kind) {       // 0 direct sum, 1 Lagrange interpolant, 2 Hermite interpolant
  return kind == 2 ? (const void*)gc::trace_lane_kernel<2>
                   : kind == 1 ? (const void*)gc::trace_lane_kernel<1> : (const void*)gc::trace_lane_kernel<0>;
}

long long lane_blocks(const gc_field* f, long long n, int kind) {
  int per_sm = 0;
  const void* fn = lane_fn(kind);
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, gc::kLaneThreads, gc::kLaneSmemBytes) != cudaSuccess || per_sm < 1)
    per_sm = 1;
  long long blocks = (n + gc::kLaneThreads - 1) / gc::kLaneThreads;
  const long long cap = (long long)f->sm_count * per_sm;
  if (blocks > cap) blocks = cap;
  return blocks < 1 ? 1 : blocks;
}

int launch_lane(const gc_field* f, gc::TraceDev& t, int kind, cudaStream_t st) {
  unsigned long long* counter = nullptr;
  GC_CUDA(cudaMallocFromPoolAsync((void**)&counter, sizeof(unsigned long long), f->pool, st));
  GC_CUDA(cudaMemsetAsync(counter, 0, sizeof(unsigned long long), st));
  t.work_counter = counter;
  const unsigned blocks = (unsigned)lane_blocks(f, t.n, kind);
  if (kind == 2) gc::trace_lane_kernel<2><<<blocks, gc::kLaneThreads, gc::kLaneSmemBytes, st>>>(f->dev, t);
  else if (kind == 1) gc::trace_lane_kernel<1><<<blocks, gc::kLaneThreads, gc::kLaneSmemBytes, st>>>(f->dev, t);
  else gc::trace_lane_kernel<0><<<blocks, gc::kLaneThreads, gc::kLaneSmemBytes, st>>>(f->dev, t);
  const cudaError_t le = cudaGetLastError();
  const cudaError_t fe = cudaFreeAsync(counter, st);          // also on a failed launch
  GC_CUDA(le);
  GC_CUDA(fe);
  return GC_OK;
}

int build_trace_dev(const gc_field* f, const gc_trace_params* p, int64_t n, gc::TraceDev* t) {
  if (!f || !p) return fail(GC_EINVAL, "gc_trace: NULL field or params");
  if (n < 0 || n > 0x7fffffffLL) return fail(GC_EINVAL, "gc_trace: n < 0 or n >= 2^31");
  if (!(p->v_ref > 0.0) || !(p->h0 > 0.0) || !(p->h_min >= 0.0) || !(p->mass > 0.0) || p->charge == 0.0 ||
      !(p->rtol >= 0.0) || !(p->atol >= 0.0) || !(p->rtol + p->atol > 0.0) || p->max_steps < 1 ||
      p->poincare_capacity < 0 || (p->flags & ~(int64_t)(GC_TRACE_RESUME | GC_TRACE_SECTION_VPAR | GC_TRACE_REFINE_LOSS)) != 0 || !std::isfinite(p->t0) || !std::isfinite(p->t_max))
    return fail(GC_EINVAL, "gc_trace: invalid integrator specification");
  t->mass = p->mass; t->charge = p->charge; t->t0 = p->t0; t->t_max = p->t_max;
  t->rtol = p->rtol; t->atol = p->atol; t->v_ref = p->v_ref; t->inv_v_ref = 1.0 / p->v_ref;
  t->h0 = p->h0; t->h_min = p->h_min; t->s_loss = p->s_loss; t->s_min = p->s_min;
  t->max_steps = p->max_steps; t->poincare_capacity = p->poincare_capacity; t->n = n;
  t->resume = (p->flags & GC_TRACE_RESUME) ? 1 : 0;
  t->section = (p->flags & GC_TRACE_SECTION_VPAR) ? 1 : 0;
  t->refine_loss = (p->flags & GC_TRACE_REFINE_LOSS) ? 1 : 0;
  return GC_OK;
}

}  // namespace

extern "C" {

const char* gc_last_error(void) { return g_last_error.c_str(); }

int gc_field_destroy(gc_field* f) {
  if (!f) return GC_OK;
  for (void* p : f->allocs) cudaFree(p);
  if (f->grid) cudaFree(f->grid);
  if (f->host_slab) cudaFree(f->host_slab);
  if (f->host_stream) cudaStreamDestroy(f->host_stream);
  if (f->pool) cudaMemPoolDestroy(f->pool);                // waits for nothing: callers synchronise before destroying
  delete f;
  return GC_OK;
}

int gc_field_create(const gc_field_desc* d, gc_field** out) {
  if (!out) return fail(GC_EINVAL, "gc_field_create: out is NULL");
  *out = nullptr;
  if (!d) return fail(GC_EINVAL, "gc_field_create: desc is NULL");
  if (d->ns < 4) return fail(GC_EINVAL, "gc_field_create: ns < 4");
  if (d->nfp < 1) return fail(GC_EINVAL, "gc_field_create: nfp < 1");
  if (d->nh < 1 || d->nk < 0) return fail(GC_EINVAL, "gc_field_create: nh < 1 or nk < 0");
  if (!d->xm || !d->xn || !d->bmnc || !d->G || !d->I || !d->iota)
    return fail(GC_EINVAL, "gc_field_create: NULL table pointer");
  if (d->nk > 0 && (!d->mode_m || !d->mode_n || !d->mode_omega || !d->mode_phase || !d->phihat))
    return fail(GC_EINVAL, "gc_field_create: NULL mode table pointer");
  if (!(d->psi0 != 0.0) || !std::isfinite(d->psi0)) return fail(GC_EINVAL, "gc_field_create: psi0 must be finite, nonzero");
  if (!all_finite(d->bmnc, (size_t)d->ns * d->nh) || !all_finite(d->G, d->ns) || !all_finite(d->I, d->ns) ||
      !all_finite(d->iota, d->ns))
    return fail(GC_EINVAL, "gc_field_create: non-finite value in an equilibrium table");
  for (const double* x : {d->bmns, d->kmnc, d->kmns})
    if (x && !all_finite(x, (size_t)d->ns * d->nh))
      return fail(GC_EINVAL, "gc_field_create: non-finite value in bmns, kmnc or kmns");
  int M = 0, N = 0;
  for (int k = 0; k < d->nh; ++k) {
    if (d->xm[k] < 0) return fail(GC_EINVAL, "gc_field_create: xm < 0");
    M = d->xm[k] > M ? d->xm[k] : M;
    const int an = d->xn[k] < 0 ? -d->xn[k] : d->xn[k];
    N = an > N ? an : N;
  }
  for (int k = 0; k < d->nk; ++k) {
    if (!(d->mode_omega[k] != 0.0) || !std::isfinite(d->mode_omega[k]))
      return fail(GC_EINVAL, "gc_field_create: mode_omega must be finite, nonzero");
    if (!std::isfinite(d->mode_phase[k])) return fail(GC_EINVAL, "gc_field_create: non-finite mode_phase");
  }
  if (d->nk > 0 && !all_finite(d->phihat, (size_t)d->ns * d->nk))
    return fail(GC_EINVAL, "gc_field_create: non-finite value in phihat");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1)
    return fail(GC_ECUDA, "gc_field_create: no CUDA device (this library has no CPU fallback)");
  gc_field* f = new (std::nothrow) gc_field;
  if (!f) return fail(GC_ENOMEM, "gc_field_create: host allocation failed");
  gc::FieldDev& v = f->dev;
  v.ns = d->ns; v.nfp = d->nfp; v.nh = d->nh; v.nk = d->nk; v.psi0 = d->psi0; v.inv_psi0 = 1.0 / d->psi0;
  v.M = M; v.N = N;
  int rc = GC_OK;
  auto up = [&](auto host, size_t count, auto** devp) {
    if (rc != GC_OK) return;
    rc = upload(host, count, devp);
    if (rc == GC_OK && *devp) f->allocs.push_back((void*)*devp);
  };
  int *xm, *xn, *mm, *mn;
  double *bmnc, *G, *I, *iota, *om, *ph, *phihat, *bmns = nullptr, *kmnc = nullptr, *kmns = nullptr;
  f->extra = d->bmns || d->kmnc || d->kmns;
  if (d->bmns) up(d->bmns, (size_t)d->ns * d->nh, &bmns);
  if (d->kmnc) up(d->kmnc, (size_t)d->ns * d->nh, &kmnc);
  if (d->kmns) up(d->kmns, (size_t)d->ns * d->nh, &kmns);
  up(d->xm, d->nh, &xm); up(d->xn, d->nh, &xn); up(d->bmnc, (size_t)d->ns * d->nh, &bmnc);
  up(d->G, d->ns, &G); up(d->I, d->ns, &I); up(d->iota, d->ns, &iota);
  up(d->mode_m, d->nk, &mm); up(d->mode_n, d->nk, &mn); up(d->mode_omega, d->nk, &om);
  std::vector<double> inv_om(d->nk);
  for (int k = 0; k < d->nk; ++k) inv_om[k] = 1.0 / d->mode_omega[k];
  double* iom = nullptr;
  up(inv_om.data(), d->nk, &iom);
  up(d->mode_phase, d->nk, &ph); up(d->phihat, (size_t)d->ns * d->nk, &phihat);
  // node rows padded to a multiple of four harmonics (field.cuh)
  double *bmnc4 = nullptr, *bmns4 = nullptr, *kmnc4 = nullptr, *kmns4 = nullptr;
  int *xmp = nullptr, *xnp = nullptr;
  const int nhp = (d->nh + 3) & ~3;
  {
    std::vector<double> pk((size_t)d->ns * nhp);
    auto pad = [&](const double* tab, double** devp) {
      if (!tab) return;
      std::fill(pk.begin(), pk.end(), 0.0);
      for (int i = 0; i < d->ns; ++i)
        std::memcpy(&pk[(size_t)i * nhp], tab + (size_t)i * d->nh, sizeof(double) * d->nh);
      up(pk.data(), pk.size(), devp);
    };
    pad(d->bmnc, &bmnc4); pad(d->bmns, &bmns4); pad(d->kmnc, &kmnc4); pad(d->kmns, &kmns4);
    std::vector<int> im(nhp, 0), in(nhp, 0);
    std::memcpy(im.data(), d->xm, sizeof(int) * d->nh);
    std::memcpy(in.data(), d->xn, sizeof(int) * d->nh);
    up(im.data(), im.size(), &xmp);
    up(in.data(), in.size(), &xnp);
  }
  if (rc == GC_OK) {
    v.bmnc4 = bmnc4; v.bmns4 = bmns4; v.kmnc4 = kmnc4; v.kmns4 = kmns4; v.xmp = xmp; v.xnp = xnp; v.nhp = nhp;
    v.xm = xm; v.xn = xn; v.bmnc = bmnc; v.G = G; v.I = I; v.iota = iota;
    v.mode_m = mm; v.mode_n = mn; v.omega = om; v.inv_omega = iom; v.phase = ph; v.phihat = phihat;
    v.bmns = bmns; v.kmnc = kmnc; v.kmns = kmns;
    rc = pack_rows(f, d);
  }
  if (rc == GC_OK) rc = pack_tile_images(f, d);
  if (rc == GC_OK) rc = pack_mma_image(f, d);
  if (rc == GC_OK) {
    int devid = 0;
    cudaGetDevice(&devid);
    cudaDeviceGetAttribute(&f->sm_count, cudaDevAttrMultiProcessorCount, devid);
    cudaMemPoolProps props{};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = devid;
    cudaError_t pe = cudaMemPoolCreate(&f->pool, &props);
    if (pe == cudaSuccess) {
      unsigned long long keep = ~0ULL;                       // never trim: the scratch is reused call after call
      pe = cudaMemPoolSetAttribute(f->pool, cudaMemPoolAttrReleaseThreshold, &keep);
    }
    if (pe != cudaSuccess) rc = fail(GC_ECUDA, std::string("cudaMemPoolCreate: ") + cudaGetErrorString(pe));
  }
  if (rc == GC_OK) {
    f->kernel = GC_KERNEL_AUTO;
    if (f->warp_ok) {
      const WarpInst* w = find_inst(f);
      rc = ensure_smem(w->trace_fn, w->smem_bytes);
      if (rc == GC_OK) rc = ensure_smem(w->rhs_fn, w->smem_bytes);
    }
  }
  if (rc != GC_OK) {
    const std::string keep = g_last_error;
    gc_field_destroy(f);
    g_last_error = keep;
    return rc;
  }
  *out = f;
  return GC_OK;
}

int gc_set_kernel(gc_field* f, int32_t kernel) {
  if (!f) return fail(GC_EINVAL, "gc_set_kernel: NULL field");
  if (kernel == GC_KERNEL_WARP && !f->warp_ok)
    return fail(GC_EINVAL, "gc_set_kernel: field does not fit the warp kernel (max|xn| <= 16, max xm <= 28, no bmns / kmnc / kmns)");
  if (kernel == GC_KERNEL_TILE && !f->tile_ok)
    return fail(GC_EINVAL, "gc_set_kernel: field does not fit the tile kernel (max|xn| <= 16, window <= 110 KB, no bmns / kmnc / kmns)");
  if (kernel == GC_KERNEL_MMA && !f->mma_ok)
    return fail(GC_EINVAL, "gc_set_kernel: field does not fit the mma kernel (max|xn| <= 16, max xm <= 16)");
  if (kernel != GC_KERNEL_AUTO && kernel != GC_KERNEL_WARP && kernel != GC_KERNEL_GENERIC && kernel != GC_KERNEL_TILE &&
      kernel != GC_KERNEL_MMA)
    return fail(GC_EINVAL, "gc_set_kernel: unknown kernel");
  f->kernel = kernel;
  return GC_OK;
}

int gc_set_option(gc_field* f, int32_t option, int64_t value) {
  if (!f) return fail(GC_EINVAL, "gc_set_option: NULL field");
  if (value < 0) return fail(GC_EINVAL, "gc_set_option: negative value");
  switch (option) {
    case GC_OPT_WAVE_PARTICLES:
      if (value != 0 && value < 4096) return fail(GC_EINVAL, "gc_set_option: a wave holds at least 4096 particles");
      f->wave_particles = value;
      return GC_OK;
    case GC_OPT_CHUNK_ATTEMPTS:
      if (value > (gc::kMmaCap > gc::kTileCap ? gc::kMmaCap : gc::kTileCap))   // the kernels' compiled maximum
        return fail(GC_EINVAL, "gc_set_option: at most " + std::to_string(gc::kMmaCap > gc::kTileCap ? gc::kMmaCap : gc::kTileCap) +
                                   " attempts per chunk (the kernels' compiled maximum)");
      f->chunk_attempts = (int)value;
      return GC_OK;
    default:
      return fail(GC_EINVAL, "gc_set_option: unknown option");
  }
}

int gc_field_set_grid(gc_field* f, int32_t ngs, int32_t nth, int32_t nze, int32_t kind, void* stream) {
  if (!f) return fail(GC_EINVAL, "gc_field_set_grid: NULL field");
  cudaStream_t st = (cudaStream_t)stream;
  // every argument is checked before the interpolant in use is touched: a refused call changes nothing
  const bool drop = ngs == 0 && nth == 0 && nze == 0;        // back to the direct harmonic sum
  if (!drop) {
    if (kind != GC_GRID_LAGRANGE && kind != GC_GRID_HERMITE) return fail(GC_EINVAL, "gc_field_set_grid: unknown kind");
    const int nmin = kind == GC_GRID_HERMITE ? 2 : 4;
    if (ngs < nmin || nth < nmin || nze < nmin)
      return fail(GC_EINVAL, "gc_field_set_grid: every node count must be >= 4 (Lagrange) / >= 2 (Hermite), or all 0");
    if (f->dev.kmnc || f->dev.kmns)
      return fail(GC_EINVAL, "gc_field_set_grid: fields with a covariant radial component K are traced by the direct sum only");
    const size_t doubles = kind == GC_GRID_HERMITE ? (size_t)ngs * (size_t)(nth + 1) * (size_t)(nze + 1) * 8
                                                   : (size_t)ngs * (size_t)(nth + 3) * (size_t)nze * 4;
    if (doubles > ((size_t)1 << 33)) return fail(GC_EINVAL, "gc_field_set_grid: table larger than 64 GiB");
  }
  if (f->grid) {                                             // drop the old interpolant
    GC_CUDA(cudaStreamSynchronize(st));
    cudaFree(f->grid);
    f->grid = nullptr;
    f->dev.grid = nullptr;
    f->dev.grid_kind = 0;
    f->dev.ngs = f->dev.nth = f->dev.nze = 0;
  }
  if (drop) return GC_OK;
  constexpr double kTwoPi = 6.283185307179586476925286766559;
  const int tb = 256;
  double* g = nullptr;
  if (kind == GC_GRID_HERMITE) {
    const size_t entries = (size_t)ngs * (size_t)(nth + 1) * (size_t)(nze + 1);
    GC_CUDA(cudaMalloc((void**)&g, entries * 8 * sizeof(double)));
    gc::grid8_build_kernel<<<(unsigned)((entries + tb - 1) / tb), tb, 0, st>>>(f->dev, ngs, nth, nze, g);
    const cudaError_t le = cudaGetLastError();
    if (le != cudaSuccess) { cudaFree(g); GC_CUDA(le); }
  } else {
    const size_t nodes = (size_t)ngs * (size_t)nth * (size_t)nze;
    const size_t total = (size_t)ngs * (size_t)(nth + 3) * (size_t)nze * 4;
    double* plain = nullptr;
    GC_CUDA(cudaMalloc((void**)&g, total * sizeof(double)));
    if (cudaMallocAsync((void**)&plain, nodes * sizeof(double), st) != cudaSuccess) {
      cudaFree(g);
      return fail(GC_ENOMEM, "gc_field_set_grid: device allocation failed");
    }
    gc::grid_build_kernel<<<(unsigned)((nodes + tb - 1) / tb), tb, 0, st>>>(f->dev, ngs, nth, nze, plain);
    gc::grid_pack_kernel<<<(unsigned)((total / 4 + tb - 1) / tb), tb, 0, st>>>(ngs, nth, nze, plain, g);
    const cudaError_t le = cudaGetLastError();
    cudaFreeAsync(plain, st);
    if (le != cudaSuccess) { cudaFree(g); GC_CUDA(le); }
  }
  // A set-up call: the table is published only once it is complete.  Traces may run on any stream (gc_trace_host
  // uses a stream of the field's own that is ordered against nothing), so the build is waited for here instead of
  // leaving every later call to order itself against `st`.
  const cudaError_t se = cudaStreamSynchronize(st);
  if (se != cudaSuccess) { cudaFree(g); GC_CUDA(se); }
  f->grid = g;
  f->dev.grid = g;
  f->dev.grid_kind = kind == GC_GRID_HERMITE ? 2 : 1;
  f->dev.ngs = ngs; f->dev.nth = nth; f->dev.nze = nze;
  f->dev.th_scale = (double)nth / kTwoPi;
  f->dev.ze_scale = (double)nze * (double)f->dev.nfp / kTwoPi;
  f->dev.inv_nth = 1.0 / (double)nth;
  f->dev.inv_nze = 1.0 / (double)nze;
  f->dev.inv_ds = (double)(ngs - 1);
  f->dev.inv_dth = f->dev.th_scale;
  f->dev.inv_dze = f->dev.ze_scale;
  return GC_OK;
}

int gc_kernel_info(const gc_field* f, int64_t n, int32_t* kernel, int32_t* blocks, int32_t* threads, int32_t* smem,
                   int32_t* regs) {
  if (!f) return fail(GC_EINVAL, "gc_kernel_info: NULL field");
  cudaFuncAttributes at{};
  int b, t, s;
  const int k = resolve_kernel(f, n);
  if (k == GC_KERNEL_MMA) {
    GC_CUDA(cudaFuncGetAttributes(&at, mma_fn(f)));
    int tsz = 0;
    b = (int)tile_geometry(f, wave_size(f, n), true, &tsz); t = gc::kMmaThreads; s = f->mma_smem;
  } else if (k == GC_KERNEL_TILE) {
    GC_CUDA(cudaFuncGetAttributes(&at, tile_fn(f)));
    int tsz = 0;
    b = (int)tile_geometry(f, wave_size(f, n), false, &tsz); t = gc::kTileThreads; s = f->tile_smem;
  } else if (k == GC_KERNEL_WARP) {
    const WarpInst* w = find_inst(f);
    GC_CUDA(cudaFuncGetAttributes(&at, w->trace_fn));
    b = f->sm_count; t = gc::kWarpsPerBlock * 32; s = w->smem_bytes;
  } else {
    const int kind = k == GC_KERNEL_GRID ? f->dev.grid_kind : 0;
    GC_CUDA(cudaFuncGetAttributes(&at, lane_fn(kind)));
    b = (int)lane_blocks(f, n, kind); t = gc::kLaneThreads; s = gc::kLaneSmemBytes;
  }
  if (kernel) *kernel = k;
  if (blocks) *blocks = b;
  if (threads) *threads = t;
  if (smem) *smem = s;
  if (regs) *regs = at.numRegs;
  return GC_OK;
}

int gc_field_eval(const gc_field* f, int64_t n, const double* s, const double* th, const double* ze, double* B,
                  double* dB, void* stream) {
  if (!f || n < 0) return fail(GC_EINVAL, "gc_field_eval: NULL field or n < 0");
  if (n == 0) return GC_OK;
  if (!s || !th || !ze || !B) return fail(GC_EINVAL, "gc_field_eval: NULL array");
  const int tb = 128;
  gc::field_eval_kernel<<<(unsigned)((n + tb - 1) / tb), tb, 0, (cudaStream_t)stream>>>(f->dev, n, s, th, ze, B, dB);
  GC_CUDA(cudaGetLastError());
  return GC_OK;
}

int gc_kcov_eval(const gc_field* f, int64_t n, const double* s, const double* th, const double* ze, double* K,
                 double* dK, void* stream) {
  if (!f || n < 0) return fail(GC_EINVAL, "gc_kcov_eval: NULL field or n < 0");
  if (n == 0) return GC_OK;
  if (!s || !th || !ze || !K) return fail(GC_EINVAL, "gc_kcov_eval: NULL array");
  const int tb = 128;
  gc::kcov_eval_kernel<<<(unsigned)((n + tb - 1) / tb), tb, 0, (cudaStream_t)stream>>>(f->dev, n, s, th, ze, K, dK);
  GC_CUDA(cudaGetLastError());
  return GC_OK;
}

int gc_pert_eval(const gc_field* f, int64_t n, const double* s, const double* th, const double* ze, double t,
                 double* out, void* stream) {
  if (!f || n < 0) return fail(GC_EINVAL, "gc_pert_eval: NULL field or n < 0");
  if (n == 0) return GC_OK;
  if (!s || !th || !ze || !out) return fail(GC_EINVAL, "gc_pert_eval: NULL array");
  const int tb = 128;
  gc::pert_eval_kernel<<<(unsigned)((n + tb - 1) / tb), tb, 0, (cudaStream_t)stream>>>(f->dev, n, s, th, ze, t, out);
  GC_CUDA(cudaGetLastError());
  return GC_OK;
}

int gc_rhs_eval(const gc_field* f, double mass, double charge, double t, int64_t n, const double* y,
                const double* mu, double* dydt, void* stream) {
  if (!f || n < 0) return fail(GC_EINVAL, "gc_rhs_eval: NULL field or n < 0");
  if (n == 0) return GC_OK;
  if (!y || !mu || !dydt) return fail(GC_EINVAL, "gc_rhs_eval: NULL array");
  const int kern = resolve_kernel(f, n);
  if (kern == GC_KERNEL_TILE || kern == GC_KERNEL_MMA) {
    gc::TraceDev td{};
    td.mass = mass; td.charge = charge; td.t0 = t; td.t_max = t; td.v_ref = 1.0; td.inv_v_ref = 1.0;
    td.n = n; td.s0 = y; td.th0 = y + n; td.ze0 = y + 2 * n; td.vpar0 = y + 3 * n; td.mu = mu;
    td.max_steps = 1;
    return launch_tile(f, td, 1, dydt, (cudaStream_t)stream, kern == GC_KERNEL_MMA);
  }
  if (kern == GC_KERNEL_WARP) {
    const WarpInst* w = find_inst(f);
    long long nn = n;
    void* args[] = {(void*)&f->dev, &mass, &charge, &t, &nn, (void*)&y, (void*)&mu, (void*)&dydt};
    long long blocks = (n + gc::kWarpsPerBlock - 1) / gc::kWarpsPerBlock;
    if (blocks > f->sm_count) blocks = f->sm_count;
    GC_CUDA(cudaLaunchKernel(w->rhs_fn, dim3((unsigned)blocks), dim3(gc::kWarpsPerBlock * 32), args,
                             (size_t)w->smem_bytes, (cudaStream_t)stream));
  } else {
    const int tb = 128;
    gc::rhs_eval_generic_kernel<<<(unsigned)((n + tb - 1) / tb), tb, 0, (cudaStream_t)stream>>>(
        f->dev, mass, charge, t, n, y, mu, dydt);
    GC_CUDA(cudaGetLastError());
  }
  return GC_OK;
}

}  // extern "C"

namespace {
int trace_common(const gc_field* f, const gc_trace_params* params, int64_t n, const double* s0, const double* th0,
                 const double* ze0, const double* vpar0, const double* mu, double* h_inout, double* y_out,
                 double* t_out, int32_t* status, int32_t* n_acc, int32_t* n_rej, int32_t* n_forced, double* poincare,
                 int64_t* poincare_count, double sample_t0, double sample_dt, int64_t nsamp, double* samples,
                 int32_t* sample_end, void* stream) {
  gc::TraceDev t{};
  int rc = build_trace_dev(f, params, n, &t);
  if (rc != GC_OK) return rc;
  if (nsamp < 0 || (nsamp > 0 && (!samples || !sample_end || !(sample_dt > 0.0) || !std::isfinite(sample_t0))))
    return fail(GC_EINVAL, "gc_trace_sampled: nsamp > 0 needs sample_dt > 0, finite sample_t0, samples and sample_end");
  if (n == 0) return GC_OK;
  if (!s0 || !th0 || !ze0 || !vpar0 || !mu || !y_out || !t_out || !status)
    return fail(GC_EINVAL, "gc_trace: NULL particle array");
  if (params->poincare_capacity > 0 && (!poincare || !poincare_count))
    return fail(GC_EINVAL, "gc_trace: poincare_capacity > 0 needs poincare and poincare_count");
  cudaStream_t st = (cudaStream_t)stream;
  t.s0 = s0; t.th0 = th0; t.ze0 = ze0; t.vpar0 = vpar0; t.mu = mu; t.h_inout = h_inout;
  t.y_out = y_out; t.t_out = t_out; t.status = status; t.n_acc = n_acc; t.n_rej = n_rej; t.n_forced = n_forced;
  t.poincare = poincare;
  t.poincare_count = reinterpret_cast<unsigned long long*>(poincare_count);
  if (!poincare || !poincare_count) t.poincare_capacity = 0;
  if (poincare_count) GC_CUDA(cudaMemsetAsync(poincare_count, 0, sizeof(int64_t), st));
  t.sample_t0 = sample_t0; t.sample_dt = sample_dt; t.nsamp = nsamp; t.samples = samples; t.sample_end = sample_end;
  int kern = resolve_kernel(f, n);
  if (kern == GC_KERNEL_WARP && (nsamp > 0 || t.section != 0 || t.refine_loss != 0))
    kern = GC_KERNEL_GENERIC;                       // the warp kernel has neither samples nor the bounce section
  if (kern == GC_KERNEL_TILE || kern == GC_KERNEL_MMA) return launch_tile(f, t, 0, nullptr, st, kern == GC_KERNEL_MMA);
  if (kern == GC_KERNEL_WARP) {
    const WarpInst* w = find_inst(f);
    unsigned long long* counter = nullptr;
    GC_CUDA(cudaMallocFromPoolAsync((void**)&counter, sizeof(unsigned long long), f->pool, st));
    GC_CUDA(cudaMemsetAsync(counter, 0, sizeof(unsigned long long), st));
    t.work_counter = counter;
    void* args[] = {(void*)&f->dev, (void*)&t};
    long long blocks = (n + gc::kWarpsPerBlock - 1) / gc::kWarpsPerBlock;
    if (blocks > f->sm_count) blocks = f->sm_count;
    const cudaError_t le = cudaLaunchKernel(w->trace_fn, dim3((unsigned)blocks), dim3(gc::kWarpsPerBlock * 32), args,
                                            (size_t)w->smem_bytes, st);
    const cudaError_t fe = cudaFreeAsync(counter, st);      // also on a failed launch
    GC_CUDA(le);
    GC_CUDA(fe);
  } else {
    return launch_lane(f, t, kern == GC_KERNEL_GRID ? f->dev.grid_kind : 0, st);
  }
  return GC_OK;
}
}  // namespace

extern "C" {

int gc_trace(const gc_field* f, const gc_trace_params* params, int64_t n, const double* s0, const double* th0,
             const double* ze0, const double* vpar0, const double* mu, double* h_inout, double* y_out,
             double* t_out, int32_t* status, int32_t* n_acc, int32_t* n_rej, int32_t* n_forced, double* poincare,
             int64_t* poincare_count, void* stream) {
  return trace_common(f, params, n, s0, th0, ze0, vpar0, mu, h_inout, y_out, t_out, status, n_acc, n_rej, n_forced,
                      poincare, poincare_count, 0.0, 0.0, 0, nullptr, nullptr, stream);
}

int gc_trace_sampled(const gc_field* f, const gc_trace_params* params, int64_t n, const double* s0, const double* th0,
                     const double* ze0, const double* vpar0, const double* mu, double* h_inout, double* y_out,
                     double* t_out, int32_t* status, int32_t* n_acc, int32_t* n_rej, int32_t* n_forced,
                     double sample_t0, double sample_dt, int64_t nsamp, double* samples, int32_t* sample_end,
                     void* stream) {
  if (params && params->poincare_capacity != 0)
    return fail(GC_EINVAL, "gc_trace_sampled: records no Poincare crossings (poincare_capacity must be 0)");
  return trace_common(f, params, n, s0, th0, ze0, vpar0, mu, h_inout, y_out, t_out, status, n_acc, n_rej, n_forced,
                      nullptr, nullptr, sample_t0, sample_dt, nsamp, samples, sample_end, stream);
}

int gc_trace_symplectic(const gc_field* f, const gc_symplectic_params* p, int64_t n, const double* s0,
                        const double* th0, const double* ze0, const double* vpar0, const double* mu,
                        const double* chi_nodes, double* y_out, double* t_out, int32_t* status, int32_t* n_steps,
                        int32_t* n_iter, int64_t sample_stride, int64_t nsamp, double* samples, int32_t* sample_end,
                        void* stream) {
  if (!f || !p) return fail(GC_EINVAL, "gc_trace_symplectic: NULL field or params");
  if (f->dev.nk > 0 || f->dev.kmnc || f->dev.kmns)
    return fail(GC_EINVAL, "gc_trace_symplectic: static fields with K = 0 only (no modes, no kmnc / kmns)");
  if (n < 0 || n > 0x7fffffffLL) return fail(GC_EINVAL, "gc_trace_symplectic: n < 0 or n >= 2^31");
  if (!(p->mass > 0.0) || p->charge == 0.0 || !(p->dt > 0.0) || !std::isfinite(p->t0) || p->nsteps < 0 ||
      !(p->newton_tol > 0.0) || p->max_iter < 1 || p->max_iter > 1000 || (p->flags & ~(int64_t)GC_TRACE_RESUME) != 0)
    return fail(GC_EINVAL, "gc_trace_symplectic: invalid integrator specification");
  if (nsamp < 0 || (nsamp > 0 && (sample_stride < 1 || !samples || !sample_end)))
    return fail(GC_EINVAL, "gc_trace_symplectic: nsamp > 0 needs sample_stride >= 1, samples and sample_end");
  if (n == 0) return GC_OK;
  if (!s0 || !th0 || !ze0 || !vpar0 || !mu || !chi_nodes || !y_out || !t_out || !status)
    return fail(GC_EINVAL, "gc_trace_symplectic: NULL particle array or chi_nodes");
  // large ensembles on the direct sum: the cell-binned mma engine (one pass = one field evaluation per lane)
  {
    const int64_t nmin = (f->dev.M <= 8 && f->dev.N <= 8) ? GC_TILE_MIN_PARTICLES_SMALL : GC_TILE_MIN_PARTICLES;
    if (!f->dev.grid && f->mma_ok && !f->extra && f->mma_blocks_per_sm > 0 && n >= nmin && nsamp == 0 &&
        p->nsteps >= 1 && f->kernel != GC_KERNEL_GENERIC) {
      gc::TraceDev t{};
      t.mass = p->mass; t.charge = p->charge; t.t0 = p->t0; t.t_max = p->t0; t.v_ref = 1.0; t.inv_v_ref = 1.0;
      t.s_loss = p->s_loss; t.s_min = p->s_min; t.max_steps = 1; t.n = n;
      t.resume = (p->flags & GC_TRACE_RESUME) ? 1 : 0;
      t.s0 = s0; t.th0 = th0; t.ze0 = ze0; t.vpar0 = vpar0; t.mu = mu;
      t.y_out = y_out; t.t_out = t_out; t.status = status; t.n_acc = n_steps; t.n_rej = n_iter;
      t.sym_dt = p->dt; t.sym_tol = p->newton_tol; t.sym_nsteps = p->nsteps; t.sym_max_iter = (int)p->max_iter;
      t.chi = chi_nodes;
      return launch_tile(f, t, 0, nullptr, (cudaStream_t)stream, true, true);
    }
  }
  gc::SymplecticDev d{};
  d.mass = p->mass; d.charge = p->charge; d.t0 = p->t0; d.dt = p->dt; d.s_loss = p->s_loss; d.s_min = p->s_min;
  d.tol = p->newton_tol; d.nsteps = p->nsteps; d.n = n; d.sample_stride = sample_stride > 0 ? sample_stride : 1;
  d.nsamp = nsamp; d.max_iter = (int)p->max_iter; d.resume = (p->flags & GC_TRACE_RESUME) ? 1 : 0;
  d.s0 = s0; d.th0 = th0; d.ze0 = ze0; d.vpar0 = vpar0; d.mu = mu; d.chi = chi_nodes;
  d.y_out = y_out; d.t_out = t_out; d.status = status; d.n_steps = n_steps; d.n_iter = n_iter;
  d.samples = samples; d.sample_end = sample_end;
  const int tb = 128;
  long long blocks = (n + tb - 1) / tb;
  if (blocks > (long long)f->sm_count * 16) blocks = (long long)f->sm_count * 16;
  if (f->dev.grid && f->dev.grid_kind == 2)
    gc::trace_symplectic_kernel<2><<<(unsigned)blocks, tb, 0, (cudaStream_t)stream>>>(f->dev, d);
  else if (f->dev.grid) gc::trace_symplectic_kernel<1><<<(unsigned)blocks, tb, 0, (cudaStream_t)stream>>>(f->dev, d);
  else gc::trace_symplectic_kernel<0><<<(unsigned)blocks, tb, 0, (cudaStream_t)stream>>>(f->dev, d);
  GC_CUDA(cudaGetLastError());
  return GC_OK;
}

int gc_pzeta_eval(const gc_field* f, double mass, double charge, int64_t n, const double* y, const double* t,
                  const double* chi_nodes, double* out, void* stream) {
  if (!f || n < 0) return fail(GC_EINVAL, "gc_pzeta_eval: NULL field or n < 0");
  if (n == 0) return GC_OK;
  if (!y || !chi_nodes || !out || charge == 0.0) return fail(GC_EINVAL, "gc_pzeta_eval: NULL array or zero charge");
  const int tb = 128;
  gc::pzeta_eval_kernel<<<(unsigned)((n + tb - 1) / tb), tb, 0, (cudaStream_t)stream>>>(f->dev, mass, charge, n, y, t,
                                                                                       chi_nodes, out);
  GC_CUDA(cudaGetLastError());
  return GC_OK;
}

int gc_birkhoff(int64_t n, int64_t nsamp, const double* series, int64_t j_first, const int32_t* sample_end,
                double* out, void* stream) {
  if (n < 0 || nsamp < 0 || j_first < 0) return fail(GC_EINVAL, "gc_birkhoff: negative size");
  if (n == 0) return GC_OK;
  if (!series || !out) return fail(GC_EINVAL, "gc_birkhoff: NULL array");
  const int tb = 128;
  gc::birkhoff_kernel<<<(unsigned)((n + tb - 1) / tb), tb, 0, (cudaStream_t)stream>>>(n, nsamp, series, j_first,
                                                                                     sample_end, out);
  GC_CUDA(cudaGetLastError());
  return GC_OK;
}

int gc_orbit_diagnostics(int64_t n, int64_t nsamp, const double* samples, int64_t j_first, const int32_t* sample_end,
                         double sample_dt, double mass, double* out, void* stream) {
  if (n < 0 || nsamp < 0 || j_first < 0) return fail(GC_EINVAL, "gc_orbit_diagnostics: negative size");
  if (!(sample_dt > 0.0) || !(mass > 0.0)) return fail(GC_EINVAL, "gc_orbit_diagnostics: sample_dt and mass must be > 0");
  if (n == 0) return GC_OK;
  if (!samples || !out) return fail(GC_EINVAL, "gc_orbit_diagnostics: NULL array");
  const int tb = 128;
  gc::orbit_diag_kernel<<<(unsigned)((n + tb - 1) / tb), tb, 0, (cudaStream_t)stream>>>(n, nsamp, samples, j_first,
                                                                                       sample_end, sample_dt, mass, out);
  GC_CUDA(cudaGetLastError());
  return GC_OK;
}

int gc_trace_host(gc_field* f, const gc_trace_params* params, int64_t n, const double* s0,
                  const double* th0, const double* ze0, const double* vpar0, const double* mu, double* h_inout,
                  double* y_out, double* t_out, int32_t* status, int32_t* n_acc, int32_t* n_rej,
                  int32_t* n_forced, double* poincare, int64_t* poincare_count) {
  if (!f || !params || n < 0) return fail(GC_EINVAL, "gc_trace_host: NULL field/params or n < 0");
  if (n == 0) return GC_OK;
  if (!s0 || !th0 || !ze0 || !vpar0 || !mu || !y_out || !t_out || !status)
    return fail(GC_EINVAL, "gc_trace_host: NULL particle array");
  const size_t nd = (size_t)n;
  const int64_t cap = (poincare && poincare_count) ? params->poincare_capacity : 0;
  // one device slab: 5 inputs, h, y_out[4], t_out (doubles) | status + 3 counters (int32) | poincare
  const size_t n_dbl = nd * 11 + (size_t)cap * 4 + 1;
  int rc = GC_OK;
  auto cleanup = [&]() {};
#define GC_H(expr)                                                                 \
  do {                                                                             \
    cudaError_t e_ = (expr);                                                       \
    if (e_ != cudaSuccess) {                                                       \
      rc = fail(e_ == cudaErrorMemoryAllocation ? GC_ENOMEM : GC_ECUDA,            \
                std::string(#expr) + ": " + cudaGetErrorString(e_));               \
      cleanup();                                                                   \
      return rc;                                                                   \
    }                                                                              \
  } while (0)
  // stream and device slab live in the field and are reused by later calls; calls on one field must not overlap
  gc_field* fm = f;
  if (fm->host_busy.exchange(true)) return fail(GC_EINVAL, "gc_trace_host: another gc_trace_host call is running on this field");
  struct Release { gc_field* f; ~Release() { f->host_busy.store(false); } } release{fm};
  if (!fm->host_stream) GC_H(cudaStreamCreateWithFlags(&fm->host_stream, cudaStreamNonBlocking));
  const size_t dbl_bytes = ((n_dbl * sizeof(double) + 255) / 256) * 256;
  const size_t need = dbl_bytes + nd * 4 * sizeof(int32_t);
  if (need > fm->host_slab_bytes) {
    if (fm->host_slab) { cudaFree(fm->host_slab); fm->host_slab = nullptr; fm->host_slab_bytes = 0; }
    GC_H(cudaMalloc(&fm->host_slab, need));
    fm->host_slab_bytes = need;
  }
  cudaStream_t st = fm->host_stream;
  double* dbl = reinterpret_cast<double*>(fm->host_slab);
  int32_t* i32 = reinterpret_cast<int32_t*>(reinterpret_cast<unsigned char*>(fm->host_slab) + dbl_bytes);
  double *d_s = dbl, *d_th = dbl + nd, *d_ze = dbl + 2 * nd, *d_v = dbl + 3 * nd, *d_mu = dbl + 4 * nd,
         *d_h = dbl + 5 * nd, *d_y = dbl + 6 * nd, *d_t = dbl + 10 * nd, *d_pc = dbl + 11 * nd;
  int64_t* d_cnt = reinterpret_cast<int64_t*>(dbl + 11 * nd + (size_t)cap * 4);
  const size_t bytes = nd * sizeof(double);
  GC_H(cudaMemcpyAsync(d_s, s0, bytes, cudaMemcpyHostToDevice, st));
  GC_H(cudaMemcpyAsync(d_th, th0, bytes, cudaMemcpyHostToDevice, st));
  GC_H(cudaMemcpyAsync(d_ze, ze0, bytes, cudaMemcpyHostToDevice, st));
  GC_H(cudaMemcpyAsync(d_v, vpar0, bytes, cudaMemcpyHostToDevice, st));
  GC_H(cudaMemcpyAsync(d_mu, mu, bytes, cudaMemcpyHostToDevice, st));
  if (h_inout) GC_H(cudaMemcpyAsync(d_h, h_inout, bytes, cudaMemcpyHostToDevice, st));
  if (params->flags & GC_TRACE_RESUME) {
    GC_H(cudaMemcpyAsync(d_y, y_out, 4 * bytes, cudaMemcpyHostToDevice, st));
    GC_H(cudaMemcpyAsync(d_t, t_out, bytes, cudaMemcpyHostToDevice, st));
    GC_H(cudaMemcpyAsync(i32, status, nd * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (n_acc) GC_H(cudaMemcpyAsync(i32 + nd, n_acc, nd * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (n_rej) GC_H(cudaMemcpyAsync(i32 + 2 * nd, n_rej, nd * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    if (n_forced) GC_H(cudaMemcpyAsync(i32 + 3 * nd, n_forced, nd * sizeof(int32_t), cudaMemcpyHostToDevice, st));
  }
  rc = gc_trace(f, params, n, d_s, d_th, d_ze, d_v, d_mu, h_inout ? d_h : nullptr, d_y, d_t, i32,
                n_acc ? i32 + nd : nullptr, n_rej ? i32 + 2 * nd : nullptr, n_forced ? i32 + 3 * nd : nullptr,
                cap > 0 ? d_pc : nullptr, cap > 0 ? d_cnt : nullptr, st);
  if (rc != GC_OK) { cleanup(); return rc; }
  GC_H(cudaMemcpyAsync(y_out, d_y, 4 * bytes, cudaMemcpyDeviceToHost, st));
  GC_H(cudaMemcpyAsync(t_out, d_t, bytes, cudaMemcpyDeviceToHost, st));
  GC_H(cudaMemcpyAsync(status, i32, nd * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (h_inout) GC_H(cudaMemcpyAsync(h_inout, d_h, bytes, cudaMemcpyDeviceToHost, st));
  if (n_acc) GC_H(cudaMemcpyAsync(n_acc, i32 + nd, nd * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (n_rej) GC_H(cudaMemcpyAsync(n_rej, i32 + 2 * nd, nd * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (n_forced) GC_H(cudaMemcpyAsync(n_forced, i32 + 3 * nd, nd * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (cap > 0) {
    GC_H(cudaMemcpyAsync(poincare_count, d_cnt, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    GC_H(cudaStreamSynchronize(st));
    const int64_t got = *poincare_count < cap ? *poincare_count : cap;
    if (got > 0) GC_H(cudaMemcpyAsync(poincare, d_pc, (size_t)got * 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
  } else if (poincare_count) {
    *poincare_count = 0;
  }
  GC_H(cudaStreamSynchronize(st));
#undef GC_H
  cleanup();
  return GC_OK;
}

}  // extern "C"

// ---- gc_trace_noalloc: the mma trace with its work area in a fixed array of the library image (include/gcorbit.h) ----
// For callers that may not allocate device memory once they run (a host application that owns the whole GPU through
// its own arena, a loop with a deadline, a plug-in whose host forbids the CUDA allocation calls).  Nothing above this
// line is changed by it; the carve-up of the work area below repeats launch_tile's on purpose.
namespace {

// The work area.  It exists once per GPU that loads the library and lives until the process ends.
static __device__ __align__(256) unsigned char g_noalloc_scratch[GC_NOALLOC_SCRATCH_BYTES];

// In host code the name g_noalloc_scratch is only a handle for the runtime, not an address the GPU understands: the
// device address has to be asked for, per GPU, with that GPU current.
constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mutex;
unsigned char* g_noalloc_addr[kNoAllocMaxDevices] = {};

int noalloc_scratch(unsigned char** out) {
  int dev = -1;
  GC_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(GC_EINVAL, "gc_trace_noalloc: device ordinal out of range");
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_addr[dev]) {                               // first call on this GPU: the set-up step
    void* p = nullptr;
    GC_CUDA(cudaGetSymbolAddress(&p, g_noalloc_scratch));
    if (!p) return fail(GC_ECUDA, "gc_trace_noalloc: cudaGetSymbolAddress returned no address");
    g_noalloc_addr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_noalloc_addr[dev];
  return GC_OK;
}

}  // namespace

extern "C" {

int gc_trace_noalloc(const gc_field* f, const gc_trace_params* params, int64_t n, const double* s0, const double* th0,
                     const double* ze0, const double* vpar0, const double* mu, double* h_inout, double* y_out,
                     double* t_out, int32_t* status, int32_t* n_acc, int32_t* n_rej, int32_t* n_forced,
                     double* poincare, int64_t* poincare_count, void* stream) {
  gc::TraceDev t{};
  int rc = build_trace_dev(f, params, n, &t);
  if (rc != GC_OK) return rc;
  if (n > GC_NOALLOC_MAX_PARTICLES)
    return fail(GC_EINVAL, "gc_trace_noalloc: n = " + std::to_string((long long)n) + " particles, the fixed work area holds " +
                               std::to_string((int)GC_NOALLOC_MAX_PARTICLES) + " (GC_NOALLOC_MAX_PARTICLES); trace the ensemble in slices");
  if (!f->mma_ok) return fail(GC_EINVAL, "gc_trace_noalloc: the field does not fit the mma kernel (max |xn| <= 16, max xm <= 16)");
  if (f->dev.grid) return fail(GC_EINVAL, "gc_trace_noalloc: the field has a 3-D interpolant set (gc_field_set_grid)");
  // the same carve-up as launch_tile: records, then order | cnt | cursor | start | tstart | ctrl | next
  const int ncell = f->dev.ns - 3;
  const size_t wn = (size_t)(n > 0 ? n : 1);                // one record slot per particle
  const size_t rec_bytes = wn * gc::kRecDoubles * sizeof(double);
  const size_t nbin = (size_t)ncell * gc::kSubBins;
  const size_t order_count = (wn + 1) & ~(size_t)1;
  const size_t zero_count = 2 * nbin + (size_t)2 * (ncell + 1) + 8 + 4;
  const size_t need = rec_bytes + (order_count + zero_count) * sizeof(int);
  if (need > (size_t)GC_NOALLOC_SCRATCH_BYTES)
    return fail(GC_EINVAL, "gc_trace_noalloc: " + std::to_string(need) + " bytes of work area needed for n = " +
                               std::to_string((long long)n) + " and ns = " + std::to_string(f->dev.ns) + ", the fixed array has " +
                               std::to_string((int)GC_NOALLOC_SCRATCH_BYTES) + " (GC_NOALLOC_SCRATCH_BYTES)");
  if (n == 0) return GC_OK;
  if (!s0 || !th0 || !ze0 || !vpar0 || !mu || !y_out || !t_out || !status)
    return fail(GC_EINVAL, "gc_trace_noalloc: NULL particle array");
  if (params->poincare_capacity > 0 && (!poincare || !poincare_count))
    return fail(GC_EINVAL, "gc_trace_noalloc: poincare_capacity > 0 needs poincare and poincare_count");
  unsigned char* slab = nullptr;
  rc = noalloc_scratch(&slab);
  if (rc != GC_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  t.s0 = s0; t.th0 = th0; t.ze0 = ze0; t.vpar0 = vpar0; t.mu = mu; t.h_inout = h_inout;
  t.y_out = y_out; t.t_out = t_out; t.status = status; t.n_acc = n_acc; t.n_rej = n_rej; t.n_forced = n_forced;
  t.poincare = poincare;
  t.poincare_count = reinterpret_cast<unsigned long long*>(poincare_count);
  if (!poincare || !poincare_count) t.poincare_capacity = 0;
  if (poincare_count) GC_CUDA(cudaMemsetAsync(poincare_count, 0, sizeof(int64_t), st));
  gc::TileScratch sc{};
  sc.slots = (long long)wn;
  sc.chunk = f->chunk_attempts;
  sc.rec = reinterpret_cast<double*>(slab);
  int* ip = reinterpret_cast<int*>(slab + rec_bytes);
  sc.order = ip; ip += order_count;
  sc.cnt = ip; ip += nbin;
  sc.cursor = ip; ip += nbin;
  sc.start = ip; ip += ncell + 1;
  sc.tstart = ip; ip += ncell + 1;
  sc.ctrl = ip; ip += 8;
  ip += ((reinterpret_cast<uintptr_t>(ip) & 7) ? 1 : 0);   // the 64-bit input cursor
  sc.next = reinterpret_cast<unsigned long long*>(ip);
  // the array keeps what the last call left in it: the bin counts, cursors, offsets, control words and the input
  // cursor must start at zero (records and `order` are written by the kernel before it reads them)
  GC_CUDA(cudaMemsetAsync(sc.cnt, 0, zero_count * sizeof(int), st));
  int per_tile = 0;
  const long long blocks = tile_geometry(f, (long long)wn, true, &per_tile);
  sc.tile_size = per_tile;
  gc::FieldDev fd = f->dev;
  int mode = 0;
  double* rhs_out = nullptr;
  void* args[] = {(void*)&fd, (void*)&t, (void*)&sc, (void*)&mode, (void*)&rhs_out};
  const bool sample = t.section != 0 || t.refine_loss != 0;   // the diagnostics build of the kernel, as in launch_tile
  GC_CUDA(cudaLaunchCooperativeKernel(mma_fn(f, sample), dim3((unsigned)blocks), dim3(gc::kMmaThreads), args,
                                      (size_t)f->mma_smem, st));
  return GC_OK;
}

}  // extern "C"
