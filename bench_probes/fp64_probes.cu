// fp64_probes.cu -- microbenchmarks of the box, built as libgcprobes.so for bench.py ONLY.  Not part of the product
// boundary (include/gcorbit.h declares none of this; libgcorbit.so does not contain it): they measure the
// denominators and the instruction costs that DESIGN.md section 6 quotes, in the run that prints the bench line.
//   gcprobe_dfma    register-only DFMA loop on every SM                        -> FP64 FLOP/s (2 per DFMA)
//   gcprobe_dmma    DMMA.8x8x4 (mma.sync.m8n8k4.f64), 8 independent accumulators per warp, alone and with one DFMA
//                   per DMMA mixed in                                          -> FLOP/s of each
//   gcprobe_lds128  LDS.128 issue cost of a warp: all lanes distinct 16-byte addresses, and even/odd lane pairs on
//                   the same 16 bytes                                          -> data-pipe cycles per warp instruction per SM
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -shared -Xcompiler -fPIC
#include <cuda_runtime.h>

namespace {

__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

__global__ void dfma_probe_kernel(double* out, int iters) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6,
         a7 = a0 + 7;
  const double x = 0.999999999, y = 1e-12;
  for (int i = 0; i < iters; ++i) {
    a0 = fma(a0, x, y); a1 = fma(a1, x, y); a2 = fma(a2, x, y); a3 = fma(a3, x, y);
    a4 = fma(a4, x, y); a5 = fma(a5, x, y); a6 = fma(a6, x, y); a7 = fma(a7, x, y);
  }
  if (a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7 == 12345.678) out[0] = a0;
}

// 8 independent DMMA.8x8x4 accumulators per warp; MIX > 0 adds MIX DFMA per 8 DMMA (the two share the FP64 units).
template <int MIX>
__global__ void dmma_probe_kernel(double* out, int iters) {
  double acc[16], f[8];
  for (int i = 0; i < 16; ++i) acc[i] = threadIdx.x * 1e-9 + i;
  for (int i = 0; i < 8; ++i) f[i] = i + 1.0;
  const double a = 0.999 + threadIdx.x * 1e-6, b = 1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < 8; ++j) dmma884(acc[2 * j], acc[2 * j + 1], a, b);
#pragma unroll
    for (int j = 0; j < MIX; ++j) f[j & 7] = fma(f[j & 7], a, b);
  }
  double s = 0.0;
  for (int i = 0; i < 16; ++i) s += acc[i];
  for (int i = 0; i < 8; ++i) s += f[i];
  if (s == 12345.678) out[0] = s;
}

// 16 LDS.128 per iteration and thread, no dependent arithmetic beyond one add per load pair.  PAIRED: lanes 2k and
// 2k + 1 read the same 16 bytes.
template <bool PAIRED>
__global__ void __launch_bounds__(256) lds_probe_kernel(double* out, int iters, long long* cycles) {
  __shared__ double2 tab[2048];
  for (int i = threadIdx.x; i < 2048; i += blockDim.x) tab[i] = make_double2(i * 1e-3, 1.0);
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const int slot = PAIRED ? (lane >> 1) : lane;
  double s0 = 0.0, s1 = 0.0;
  const long long c0 = clock64();
  for (int it = 0; it < iters; ++it) {
    const double2* p = tab + ((it & 3) * 512) + slot;
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const double2 v = p[j * 32];
      s0 += v.x;
      s1 += v.y;
    }
  }
  const long long c1 = clock64();
  if (threadIdx.x == 0 && blockIdx.x == 0) cycles[0] = c1 - c0;
  if (s0 + s1 == 12345.678) out[0] = s0;
}

template <class F>
cudaError_t best_of(int reps, float* best, F launch) {
  cudaEvent_t a, b;
  cudaError_t e = cudaEventCreate(&a);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&b);
  if (e != cudaSuccess) return e;
  *best = 1e30f;
  for (int rep = 0; rep < reps + 1; ++rep) {                          // first repetition warms up
    cudaEventRecord(a);
    launch();
    cudaEventRecord(b);
    e = cudaEventSynchronize(b);
    if (e != cudaSuccess) break;
    float ms = 0;
    cudaEventElapsedTime(&ms, a, b);
    if (rep > 0 && ms < *best) *best = ms;
  }
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  return e != cudaSuccess ? e : cudaGetLastError();
}

int sm_count() {
  int devid = 0, sms = 0;
  if (cudaGetDevice(&devid) != cudaSuccess) return 0;
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, devid);
  return sms;
}

}  // namespace

extern "C" {

// Returns 0 or a cudaError_t.  *flops_per_s: 2 flop per DFMA.
int gcprobe_dfma(double* flops_per_s, double* elapsed_ms) {
  const int sms = sm_count();
  if (sms < 1) return (int)cudaErrorNoDevice;
  double* out = nullptr;
  cudaError_t e = cudaMalloc((void**)&out, sizeof(double));
  if (e != cudaSuccess) return (int)e;
  const int iters = 200000, blocks = sms * 2, threads = 512;
  float best = 0;
  e = best_of(3, &best, [&] { dfma_probe_kernel<<<blocks, threads>>>(out, iters); });
  cudaFree(out);
  if (e != cudaSuccess) return (int)e;
  if (flops_per_s) *flops_per_s = 2.0 * 8.0 * (double)iters * blocks * threads / (best * 1e-3);
  if (elapsed_ms) *elapsed_ms = best;
  return 0;
}

int gcprobe_dmma(double* flops_dmma, double* flops_mixed) {
  const int sms = sm_count();
  if (sms < 1) return (int)cudaErrorNoDevice;
  double* out = nullptr;
  cudaError_t e = cudaMalloc((void**)&out, sizeof(double));
  if (e != cudaSuccess) return (int)e;
  const int iters = 40000, blocks = sms * 2, threads = 128;           // 2 warps per SM sub-partition
  float b0 = 0, b1 = 0;
  e = best_of(3, &b0, [&] { dmma_probe_kernel<0><<<blocks, threads>>>(out, iters); });
  if (e == cudaSuccess) e = best_of(3, &b1, [&] { dmma_probe_kernel<8><<<blocks, threads>>>(out, iters); });
  cudaFree(out);
  if (e != cudaSuccess) return (int)e;
  const double warps = (double)blocks * threads / 32.0;
  if (flops_dmma) *flops_dmma = 8.0 * 512.0 * iters * warps / (b0 * 1e-3);
  if (flops_mixed) *flops_mixed = (8.0 * 512.0 + 8.0 * 64.0) * iters * warps / (b1 * 1e-3);
  return 0;
}

// SM cycles per warp-wide LDS.128 with 8 warps per SM issuing back to back (one block of 256 threads per SM):
// cycles_distinct = every lane its own 16 bytes, cycles_paired = lane pairs share 16 bytes.
int gcprobe_lds128(double* cycles_distinct, double* cycles_paired) {
  const int sms = sm_count();
  if (sms < 1) return (int)cudaErrorNoDevice;
  double* out = nullptr;
  long long* cyc = nullptr;
  cudaError_t e = cudaMalloc((void**)&out, sizeof(double));
  if (e != cudaSuccess) return (int)e;
  e = cudaMalloc((void**)&cyc, sizeof(long long));
  if (e != cudaSuccess) { cudaFree(out); return (int)e; }
  const int iters = 20000, threads = 256;
  long long c[2] = {0, 0};
  for (int which = 0; which < 2 && e == cudaSuccess; ++which) {
    for (int rep = 0; rep < 2; ++rep) {
      if (which == 0) lds_probe_kernel<false><<<sms, threads>>>(out, iters, cyc);
      else lds_probe_kernel<true><<<sms, threads>>>(out, iters, cyc);
      e = cudaDeviceSynchronize();
      if (e != cudaSuccess) break;
    }
    if (e == cudaSuccess) e = cudaMemcpy(&c[which], cyc, sizeof(long long), cudaMemcpyDeviceToHost);
  }
  cudaFree(out);
  cudaFree(cyc);
  if (e != cudaSuccess) return (int)e;
  const double instr = 16.0 * iters * (threads / 32);                 // warp instructions issued on one SM
  if (cycles_distinct) *cycles_distinct = (double)c[0] / instr;
  if (cycles_paired) *cycles_paired = (double)c[1] / instr;
  return 0;
}

}  // extern "C"
