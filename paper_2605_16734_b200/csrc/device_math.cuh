// device_math.cuh -- FP64 device helpers shared by the gcorbit kernels (sm_100a).
//
// Radial cubic Lagrange weights (O1; "Lagrange interpolation is used to evaluate the field
// throughout the volume"), argument reduction and a branch-light sin/cos pair, the Dormand-Prince 5(4)
// coefficients (O5) and the step-size factors of the controller (O6).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gc {

// ---- Dormand-Prince 5(4) coefficients (O5) ------------------------------------------------------------
namespace dp {
constexpr double c2 = 1.0 / 5.0, c3 = 3.0 / 10.0, c4 = 4.0 / 5.0, c5 = 8.0 / 9.0;
constexpr double a21 = 1.0 / 5.0;
constexpr double a31 = 3.0 / 40.0, a32 = 9.0 / 40.0;
constexpr double a41 = 44.0 / 45.0, a42 = -56.0 / 15.0, a43 = 32.0 / 9.0;
constexpr double a51 = 19372.0 / 6561.0, a52 = -25360.0 / 2187.0, a53 = 64448.0 / 6561.0, a54 = -212.0 / 729.0;
constexpr double a61 = 9017.0 / 3168.0, a62 = -355.0 / 33.0, a63 = 46732.0 / 5247.0, a64 = 49.0 / 176.0,
                 a65 = -5103.0 / 18656.0;
constexpr double a71 = 35.0 / 384.0, a73 = 500.0 / 1113.0, a74 = 125.0 / 192.0, a75 = -2187.0 / 6784.0,
                 a76 = 11.0 / 84.0;
constexpr double e1 = 71.0 / 57600.0, e3 = -71.0 / 16695.0, e4 = 71.0 / 1920.0, e5 = -17253.0 / 339200.0,
                 e6 = 22.0 / 525.0, e7 = -1.0 / 40.0;
constexpr double d1 = -12715105075.0 / 11282082432.0, d3 = 87487479700.0 / 32700410799.0,
                 d4 = -10690763975.0 / 1880347072.0, d5 = 701980252875.0 / 199316789632.0,
                 d6 = -1453857185.0 / 822651844.0, d7 = 69997945.0 / 29380423.0;
}  // namespace dp

// ---- controller (O6): S = 0.9, exponent 1/5, factors clamped to [0.2, 10] ------------------------------
constexpr double kSafety = 0.9, kMinScale = 0.2, kMaxScale = 10.0;

__device__ __forceinline__ double err_pow_m02(double err) {
  // err^(-1/5) = exp2(-log2(err)/5); err > 0 finite.  Rounding of pow differs from the host libm by ulps,
  // which moves h by ulps only ("where floating point decides").
  return pow(err, -0.2);
}

__device__ __forceinline__ double scale_after_accept(double err) {
  if (err == 0.0) return kMaxScale;
  double sc = kSafety * err_pow_m02(err);
  return fmin(fmax(sc, kMinScale), kMaxScale);
}

__device__ __forceinline__ double scale_after_reject(double err) {
  if (!isfinite(err)) return kMinScale;
  return fmax(kSafety * err_pow_m02(err), kMinScale);
}

// ---- O1: stencil start and weights, in the textbook form (used by the generic kernel) -------------------
__device__ __forceinline__ int stencil_start(int ns, double u) {
  double c = floor(u);
  if (!(c >= 1.0)) return 0;                       // also NaN
  if (c - 1.0 >= (double)(ns - 4)) return ns - 4;
  return (int)c - 1;
}

__device__ __forceinline__ void lagrange_weights(int ns, double s, int& i0, double w[4], double dw[4]) {
  const double u = s * (double)(ns - 1);
  i0 = stencil_start(ns, u);
  const double x = u - (double)i0, x1 = x - 1.0, x2 = x - 2.0, x3 = x - 3.0;
  const double sc = (double)(ns - 1);
  w[0] = -(x1 * x2 * x3) * (1.0 / 6.0);
  w[1] = (x * x2 * x3) * 0.5;
  w[2] = -(x * x1 * x3) * 0.5;
  w[3] = (x * x1 * x2) * (1.0 / 6.0);
  dw[0] = -(x2 * x3 + x1 * x3 + x1 * x2) * (sc / 6.0);
  dw[1] = (x2 * x3 + x * x3 + x * x2) * (sc * 0.5);
  dw[2] = -(x1 * x3 + x * x3 + x * x1) * (sc * 0.5);
  dw[3] = (x1 * x2 + x * x2 + x * x1) * (sc / 6.0);
}

// ---- trigonometry ------------------------------------------------------------------------------------
// a - 2 pi rint(a / 2 pi) with a two-term split of 2 pi; exact to an ulp of the result for |a| < 2^40.
__device__ __forceinline__ double reduce_2pi(double a) {
  constexpr double kInv2Pi = 0.15915494309189533576888376337251;
  constexpr double k2PiHi = 6.283185307179586232;        // double nearest 2 pi
  constexpr double k2PiLo = 2.4492935982947064e-16;      // 2 pi - k2PiHi
  const double k = rint(a * kInv2Pi);
  double r = fma(-k, k2PiHi, a);
  return fma(-k, k2PiLo, r);
}

// sin and cos of x for |x| <= ~1e5 (callers reduce first): quadrant reduction with a two-term pi/2, then
// Taylor polynomials on [-pi/4, pi/4] (truncation < 3e-18).  No table, no local memory, no slow path.
__device__ __forceinline__ void sincos_poly(double x, double& sn, double& cs) {
  constexpr double k2OverPi = 0.63661977236758134307553505349006;
  constexpr double kPio2Hi = 1.5707963267948965580;      // double nearest pi/2
  constexpr double kPio2Lo = 6.1232339957367660e-17;     // pi/2 - kPio2Hi
  const double q = rint(x * k2OverPi);
  double y = fma(-q, kPio2Hi, x);
  y = fma(-q, kPio2Lo, y);
  const int iq = (int)q;
  const double z = y * y;
  double ps = 1.0 / 355687428096000.0;                   // 1/17!
  ps = fma(ps, z, -1.0 / 1307674368000.0);               // -1/15!
  ps = fma(ps, z, 1.0 / 6227020800.0);                   // 1/13!
  ps = fma(ps, z, -1.0 / 39916800.0);                    // -1/11!
  ps = fma(ps, z, 1.0 / 362880.0);                       // 1/9!
  ps = fma(ps, z, -1.0 / 5040.0);                        // -1/7!
  ps = fma(ps, z, 1.0 / 120.0);                          // 1/5!
  ps = fma(ps, z, -1.0 / 6.0);                           // -1/3!
  const double s0 = fma(y * z, ps, y);
  double pc = 1.0 / 20922789888000.0;                    // 1/16!
  pc = fma(pc, z, -1.0 / 87178291200.0);                 // -1/14!
  pc = fma(pc, z, 1.0 / 479001600.0);                    // 1/12!
  pc = fma(pc, z, -1.0 / 3628800.0);                     // -1/10!
  pc = fma(pc, z, 1.0 / 40320.0);                        // 1/8!
  pc = fma(pc, z, -1.0 / 720.0);                         // -1/6!
  pc = fma(pc, z, 1.0 / 24.0);                           // 1/4!
  const double c0 = fma(z * z, pc, fma(-0.5, z, 1.0));
  // quadrant: iq mod 4 = 0: (s,c); 1: (c,-s); 2: (-s,-c); 3: (-c,s)
  const bool swap = iq & 1;
  double ss = swap ? c0 : s0;
  double cc = swap ? s0 : c0;
  if (iq & 2) ss = -ss;
  if ((iq + 1) & 2) cc = -cc;
  sn = ss;
  cs = cc;
}

__device__ __forceinline__ bool finite4(double a, double b, double c, double d) {
  return isfinite(a) && isfinite(b) && isfinite(c) && isfinite(d);
}

}  // namespace gc
