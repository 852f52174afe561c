// kernels_warp.cuh -- the hot-path kernel: persistent, one warp per particle, FP64, sm_100a.
//
// Layout.  With c_k = cos(k theta), s_k = sin(k theta), C_n = cos(n nfp zeta),
// S_n = sin(n nfp zeta) the harmonic sum of O2 factorises over the pairs (m, +n), (m, -n):
//     b(m,n) cos(m th - n ph) + b(m,-n) cos(m th + n ph) = P c_m C_n + Q s_m S_n,
//     P = b(m,n) + b(m,-n),  Q = b(m,n) - b(m,-n)                     (built once by gc_field_create)
// A lane owns one COLUMN (n >= 1, type P or Q): its toroidal factor (C_n or S_n) is fixed for the whole
// right-hand side, and it walks the ROWS m = 0..M, whose poloidal factors (c_m, s_m) are warp-uniform.
// Radial interpolation commutes with the sums, so the inner loop carries no interpolation at all:
//     R1[a] += A1_m * T[a][m],  R3[a] += A2_m * T[a][m]        a = 0..3 radial stencil slots
// (8 DFMA per table entry), and the 4-point Lagrange weights are applied to R1, R3 once per evaluation.
// The four table rows of the stencil live in REGISTERS (and, past NREG iterations, in lane-private shared
// memory) in a ring indexed by node mod 4, so that a particle drifting across a radial node reloads one
// row, not four.  The n = 0 column, the profiles G, I, iota and the mode amplitudes ride in the "extra"
// iterations, where a lane owns one radial table instead of one column.
//
// The integrator state is component-parallel: lane (l & 3) holds component l & 3 of y and of k1..k7, so each
// Dormand-Prince stage combination is one DFMA for all four components.
#pragma once
#include "device_math.cuh"
#include "field.cuh"
#include "kernels_generic.cuh"   // Profiles, gc_algebra, Dense3, poincare_emit

namespace gc {

constexpr int kWarpsPerBlock = 8;
constexpr int kMaxRowsM = 36;          // poloidal table entries per warp (>= NIT_MAIN * groups)
constexpr int kMaxN = 16;

constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(kFull, v, src); }
__device__ __forceinline__ double shfl_xor_d(double v, int m) { return __shfl_xor_sync(kFull, v, m); }

// Sum NV values (NV in {4, 16}) over the 32 lanes with a transposing butterfly: each round halves the
// number of values a lane still carries, so the whole reduction costs NV/2 + NV/4 + ... exchanges.
// Result: v[0] on lane group g = lane >> (5 - log2 NV) holds the total of quantity g ... then broadcast.
template <int NV>
__device__ __forceinline__ void warp_sum_bcast(double (&v)[NV], int lane) {
  static_assert(NV == 4 || NV == 16, "NV");
  constexpr int LOGV = (NV == 4) ? 2 : 4;
  // rounds with exchange (value count halves): masks 16, 8, (4, 2)
#pragma unroll
  for (int r = 0; r < LOGV; ++r) {
    const int mask = 16 >> r;
    const int half = NV >> (r + 1);
    const bool upper = lane & mask;
#pragma unroll
    for (int i = 0; i < half; ++i) {
      const double keep = upper ? v[i + half] : v[i];
      const double send = upper ? v[i] : v[i + half];
      v[i] = keep + shfl_xor_d(send, mask);
    }
  }
  // remaining rounds: plain butterfly on the single value left
#pragma unroll
  for (int r = LOGV; r < 5; ++r) v[0] += shfl_xor_d(v[0], 16 >> r);
  // lane now holds the total of quantity q(lane) = top LOGV bits of lane, bit-reversed order of selection:
  // round r chose index bit (LOGV-1-r) from lane bit (4-r)  => q = lane >> (5 - LOGV)
  const double mine = v[0];
#pragma unroll
  for (int q = 0; q < NV; ++q) v[q] = shfl_d(mine, q << (5 - LOGV));
}

template <int NIT, int NREG>
struct RowWindow {
  static constexpr int NSM = NIT - NREG;
  double reg[NREG > 0 ? NREG : 1][4];
  double* sm;   // lane-private: sm[((it - NREG) * 4 + slot) * 32]  (pointer already offset by lane)

  template <int SLOT>
  __device__ __forceinline__ void load_slot(const double* __restrict__ rows, int node, int lane) {
    const double* src = rows + (size_t)node * (NIT * 32) + lane;
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
      const double val = __ldg(src + it * 32);
      if (it < NREG) reg[it][SLOT] = val;
      else sm[((it - NREG) * 4 + SLOT) * 32] = val;
    }
  }
  __device__ __forceinline__ void load_node(const double* __restrict__ rows, int node, int lane) {
    switch (node & 3) {
      case 0: load_slot<0>(rows, node, lane); break;
      case 1: load_slot<1>(rows, node, lane); break;
      case 2: load_slot<2>(rows, node, lane); break;
      default: load_slot<3>(rows, node, lane); break;
    }
  }
  template <int IT, int SLOT>
  __device__ __forceinline__ double get() const {
    if constexpr (IT < NREG) return reg[IT][SLOT];
    else return sm[((IT - NREG) * 4 + SLOT) * 32];
  }
};

// Per-warp scratch in shared memory.
struct WarpScratch {
  double tabM[kMaxRowsM][4];     // {c_m, -m s_m, s_m, m c_m}
  double tabN[kMaxN + 1][2];     // {C_n, S_n}
};

// Everything a lane keeps for the particle it is helping with.
struct LaneRole {
  int type;        // 0 = P column, 1 = Q column
  int n;           // toroidal index of the column (>= 1); 0 if the lane has no column
  int grp;         // m-group of the lane
  double nnfp;     // n * nfp, 0 for idle lanes
};

template <int NIT_MAIN, int NX, bool MODES, int NREG>
struct WarpRhs {
  static constexpr int NIT = NIT_MAIN + NX;
  RowWindow<NIT, NREG> win;
  int cur_i0;
  double inv_mass, inv_charge;        // set once per kernel by the caller (loop-invariant reciprocals)

  // Warp-cooperative right-hand side.  All arguments and results are warp-uniform.
  __device__ __forceinline__ void operator()(const FieldDev& f, WarpScratch& sc, const LaneRole& role,
                                             int lane, double mass, double charge, double mu, double v_ref,
                                             double inv_v_ref, double t, double s, double th, double ze,
                                             double u, double dy[4]) {
    // ---- O1: stencil, ring reload, slot weights ------------------------------------------------------
    const double us = s * (double)(f.ns - 1);
    const int i0 = stencil_start(f.ns, us);
    if (i0 != cur_i0) {
      int first = i0, count = 4;
      const int d = i0 - cur_i0;
      if (cur_i0 >= 0 && d > 0 && d < 4) { first = cur_i0 + 4; count = d; }
      else if (cur_i0 >= 0 && d < 0 && d > -4) { first = i0; count = -d; }
      for (int q = 0; q < count; ++q) win.load_node(f.rows, first + q, lane);
      cur_i0 = i0;
    }
    double w[4], dw[4];
    {
      double dd[4], cden[4];
#pragma unroll
      for (int a = 0; a < 4; ++a) {
        const int j = (a - i0) & 3;                       // position of slot a inside the stencil
        dd[a] = us - (double)(i0 + j);
        cden[a] = (j == 0) ? -1.0 / 6.0 : (j == 1) ? 0.5 : (j == 2) ? -0.5 : 1.0 / 6.0;
      }
      const double p01 = dd[0] * dd[1], p23 = dd[2] * dd[3];
      const double s01 = dd[0] + dd[1], s23 = dd[2] + dd[3];
      const double scl = (double)(f.ns - 1);
      w[0] = cden[0] * (dd[1] * p23);
      w[1] = cden[1] * (dd[0] * p23);
      w[2] = cden[2] * (p01 * dd[3]);
      w[3] = cden[3] * (p01 * dd[2]);
      dw[0] = cden[0] * scl * fma(dd[1], s23, p23);       // d/du of d1 d2 d3
      dw[1] = cden[1] * scl * fma(dd[0], s23, p23);
      dw[2] = cden[2] * scl * fma(dd[3], s01, p01);
      dw[3] = cden[3] * scl * fma(dd[2], s01, p01);
    }

    // ---- a3: trig basis, one sincos per lane -----------------------------------------------------------
    const double thr = reduce_2pi(th);
    const double phr = reduce_2pi((double)f.nfp * ze);
    for (int base = 0; base < f.M + f.N; base += 32) {
      const int j = base + lane;
      if (j < f.M + f.N) {
        const bool is_m = j < f.M;
        const int k = is_m ? j + 1 : j - f.M + 1;
        double sn, cs;
        sincos_poly((double)k * (is_m ? thr : phr), sn, cs);
        if (is_m) {
          const double kd = (double)k;
          double4 e = make_double4(cs, -kd * sn, sn, kd * cs);
          *reinterpret_cast<double4*>(&sc.tabM[k][0]) = e;
        } else {
          *reinterpret_cast<double2*>(&sc.tabN[k][0]) = make_double2(cs, sn);
        }
      }
    }
    __syncwarp();

    // ---- extra iterations: n = 0 column, profiles, mode amplitudes ---------------------------------------
    double accB = 0.0, accBs = 0.0, accBth = 0.0;
    Profiles pr;
    double pv[16];                                         // B, Bs, Bth, Bze, then the 9 perturbation sums
#pragma unroll
    for (int q = 0; q < 16; ++q) pv[q] = 0.0;
    {
      double xv[NX], xd[NX];
      xv[0] = fma(w[3], win.template get<NIT_MAIN, 3>(), fma(w[2], win.template get<NIT_MAIN, 2>(),
              fma(w[1], win.template get<NIT_MAIN, 1>(), w[0] * win.template get<NIT_MAIN, 0>())));
      xd[0] = fma(dw[3], win.template get<NIT_MAIN, 3>(), fma(dw[2], win.template get<NIT_MAIN, 2>(),
              fma(dw[1], win.template get<NIT_MAIN, 1>(), dw[0] * win.template get<NIT_MAIN, 0>())));
      if constexpr (NX > 1) {
        xv[1] = fma(w[3], win.template get<NIT_MAIN + NX - 1, 3>(), fma(w[2], win.template get<NIT_MAIN + NX - 1, 2>(),
                fma(w[1], win.template get<NIT_MAIN + NX - 1, 1>(), w[0] * win.template get<NIT_MAIN + NX - 1, 0>())));
        xd[1] = fma(dw[3], win.template get<NIT_MAIN + NX - 1, 3>(), fma(dw[2], win.template get<NIT_MAIN + NX - 1, 2>(),
                fma(dw[1], win.template get<NIT_MAIN + NX - 1, 1>(), dw[0] * win.template get<NIT_MAIN + NX - 1, 0>())));
      }
      if (lane <= f.M) {                                   // n = 0 column: lane = m
        const double4 e = *reinterpret_cast<const double4*>(&sc.tabM[lane][0]);
        accB = e.x * xv[0];
        accBs = e.x * xd[0];
        accBth = e.y * xv[0];
      }
      const int lp = f.M + 1;
      pr.G = shfl_d(xv[0], lp);      pr.Gs = shfl_d(xd[0], lp);
      pr.I = shfl_d(xv[0], lp + 1);  pr.Is = shfl_d(xd[0], lp + 1);
      pr.io = shfl_d(xv[0], lp + 2); pr.ios = shfl_d(xd[0], lp + 2);
      if constexpr (MODES) {
        // mode k sits at extra index M + 4 + k
        const double zer = reduce_2pi(ze);
        const double GI = pr.G + pr.io * pr.I, GI_s = pr.Gs + pr.ios * pr.I + pr.io * pr.Is;
#pragma unroll
        for (int x = 0; x < NX; ++x) {
          const int k = x * 32 + lane - (f.M + 4);
          if (k >= 0 && k < f.nk) {
            const double ph = xv[x], ph_s = xd[x];
            const double m = (double)__ldg(f.mode_m + k), n = (double)__ldg(f.mode_n + k);
            const double om = __ldg(f.omega + k);
            const double wt = reduce_2pi(om * t);
            double sn, cs;
            sincos_poly(fma(m, thr, fma(-n, zer, wt + __ldg(f.phase + k))), sn, cs);
            const double inv = 1.0 / (om * GI);
            const double Nk = fma(pr.io, m, -n);
            const double ah = -ph * Nk * inv;
            const double ah_s = -(ph_s * Nk + ph * pr.ios * m) * inv + ph * Nk * inv * (GI_s / GI);
            pv[4] += ph * sn;
            pv[5] += ph_s * sn;
            pv[6] += m * ph * cs;
            pv[7] += -n * ph * cs;
            pv[8] += ah * sn;
            pv[9] += ah_s * sn;
            pv[10] += m * ah * cs;
            pv[11] += -n * ah * cs;
            pv[12] += om * ah * cs;
          }
        }
      }
    }

    // ---- a4: the harmonic sum, 8 DFMA per table entry ----------------------------------------------------
    double R1[4] = {0.0, 0.0, 0.0, 0.0}, R3[4] = {0.0, 0.0, 0.0, 0.0};
    {
      const int groups = 32 >> f.cl_log;
      const double* tp = &sc.tabM[role.grp][2 * role.type];
      const int stride = groups * 4;
      main_loop<0>(tp, stride, R1, R3);
    }
    const double2 tn = *reinterpret_cast<const double2*>(&sc.tabN[role.n][0]);
    const double t1 = role.n == 0 ? 0.0 : (role.type ? tn.y : tn.x);                      // C_n | S_n
    const double t2 = role.type ? role.nnfp * tn.x : -role.nnfp * tn.y;                   // d/dzeta of it
    const double S1 = fma(w[3], R1[3], fma(w[2], R1[2], fma(w[1], R1[1], w[0] * R1[0])));
    const double S2 = fma(dw[3], R1[3], fma(dw[2], R1[2], fma(dw[1], R1[1], dw[0] * R1[0])));
    const double S3 = fma(w[3], R3[3], fma(w[2], R3[2], fma(w[1], R3[1], w[0] * R3[0])));
    pv[0] = fma(t1, S1, accB);
    pv[1] = fma(t1, S2, accBs);
    pv[2] = fma(t1, S3, accBth);
    pv[3] = t2 * S1;
    __syncwarp();                                          // tabM / tabN are rewritten by the next call

    // ---- reduce over lanes, then the guiding-centre algebra (O4) -----------------------------------------
    double pt[9];
    if constexpr (MODES) {
      warp_sum_bcast<16>(pv, lane);
      pt[0] = pv[4]; pt[1] = pv[5] * f.inv_psi0; pt[2] = pv[6]; pt[3] = pv[7];
      pt[4] = pv[8]; pt[5] = pv[9] * f.inv_psi0; pt[6] = pv[10]; pt[7] = pv[11]; pt[8] = pv[12];
    } else {
      double q4[4] = {pv[0], pv[1], pv[2], pv[3]};
      warp_sum_bcast<4>(q4, lane);
      pv[0] = q4[0]; pv[1] = q4[1]; pv[2] = q4[2]; pv[3] = q4[3];
#pragma unroll
      for (int q = 0; q < 9; ++q) pt[q] = 0.0;
    }
    const double fb[4] = {pv[0], pv[1], pv[2], pv[3]};
    gc_algebra_r(mass, charge, inv_mass, inv_charge, mu, f.inv_psi0, u * v_ref, fb, pr, pt, dy);
    dy[3] *= inv_v_ref;
  }

  template <int IT>
  __device__ __forceinline__ void main_loop(const double* tp, int stride, double (&R1)[4], double (&R3)[4]) {
    if constexpr (IT < NIT_MAIN) {
      const double2 A = *reinterpret_cast<const double2*>(tp + IT * stride);
      R1[0] = fma(A.x, win.template get<IT, 0>(), R1[0]);
      R1[1] = fma(A.x, win.template get<IT, 1>(), R1[1]);
      R1[2] = fma(A.x, win.template get<IT, 2>(), R1[2]);
      R1[3] = fma(A.x, win.template get<IT, 3>(), R1[3]);
      R3[0] = fma(A.y, win.template get<IT, 0>(), R3[0]);
      R3[1] = fma(A.y, win.template get<IT, 1>(), R3[1]);
      R3[2] = fma(A.y, win.template get<IT, 2>(), R3[2]);
      R3[3] = fma(A.y, win.template get<IT, 3>(), R3[3]);
      main_loop<IT + 1>(tp, stride, R1, R3);
    }
  }
};

__device__ __forceinline__ LaneRole make_role(const FieldDev& f, int lane) {
  LaneRole r;
  const int cl = 1 << f.cl_log;
  const int c = lane & (cl - 1);
  r.grp = lane >> f.cl_log;
  r.type = c & 1;
  const int n = (c >> 1) + 1;
  r.n = (n <= f.N) ? n : 0;
  r.nnfp = (double)(r.n * f.nfp);
  return r;
}

__device__ __forceinline__ void init_scratch(WarpScratch& sc, int lane) {
  for (int i = lane; i < kMaxRowsM * 4; i += 32) (&sc.tabM[0][0])[i] = 0.0;
  for (int i = lane; i < (kMaxN + 1) * 2; i += 32) (&sc.tabN[0][0])[i] = 0.0;
  __syncwarp();
  if (lane == 0) sc.tabM[0][0] = 1.0;                      // m = 0: c_0 = 1, everything else 0
  __syncwarp();
}

extern __shared__ __align__(16) unsigned char gc_dyn_smem[];

template <int NIT_MAIN, int NX, bool MODES, int NREG>
__device__ __forceinline__ double* warp_window_smem(int warp, int lane) {
  constexpr int NSM = NIT_MAIN + NX - NREG;
  double* base = reinterpret_cast<double*>(gc_dyn_smem + sizeof(WarpScratch) * kWarpsPerBlock);
  return base + (size_t)warp * (NSM * 4 * 32) + lane;
}

// ---- the persistent trace kernel ----------------------------------------------------------------------------
template <int NIT_MAIN, int NX, bool MODES, int NREG>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 1) trace_warp_kernel(FieldDev f, TraceDev p) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  WarpScratch& sc = reinterpret_cast<WarpScratch*>(gc_dyn_smem)[warp];
  init_scratch(sc, lane);
  const LaneRole role = make_role(f, lane);
  WarpRhs<NIT_MAIN, NX, MODES, NREG> rhs;
  rhs.win.sm = warp_window_smem<NIT_MAIN, NX, MODES, NREG>(warp, lane);
  rhs.inv_mass = 1.0 / p.mass;
  rhs.inv_charge = 1.0 / p.charge;
  const int comp = lane & 3;
  constexpr double kTwoPi = 6.283185307179586476925286766559;

  for (;;) {
    // a1 / a10: pull the next particle from the queue
    unsigned long long idx = 0;
    if (lane == 0) idx = atomicAdd(p.work_counter, 1ULL);
    idx = __shfl_sync(kFull, idx, 0);
    if ((long long)idx >= p.n) break;
    const long long i = (long long)idx;
    if (p.resume && p.status[i] != 0) continue;            // finished in an earlier segment
    rhs.cur_i0 = -1000;                                    // forces a full window load

    const double mu = p.mu[i];
    // component-parallel state: lane holds component `comp`
    const double* src = comp == 0 ? p.s0 : comp == 1 ? p.th0 : comp == 2 ? p.ze0 : p.vpar0;
    double y = src[i];
    if (comp == 3) y *= p.inv_v_ref;
    double t = p.t0;
    double h = (p.h_inout && p.h_inout[i] > 0.0) ? p.h_inout[i] : p.h0;
    if (h < p.h_min) h = p.h_min;
    long long attempts = 0;
    int n_acc = 0, n_rej = 0, n_forced = 0, st = -1;
    bool prev_rejected = false, clipped = false, forced = false;
    double k1 = 0.0, k2 = 0.0, k3 = 0.0, k4 = 0.0, k5 = 0.0, k6 = 0.0, k7 = 0.0, yn = y, h_try = h;
    // One copy of the right-hand side in the instruction stream: the seven stages (and the initial k1
    // evaluation, stage 0) run through the same loop body; `stage` is warp-uniform.
    int stage = 0;
#pragma unroll 1
    while (st < 0) {
      double ys, ts;
      switch (stage) {
        case 0: ys = y; ts = t; break;
        case 1:
          h_try = h;
          clipped = false;
          if (t + h_try >= p.t_max) { h_try = p.t_max - t; clipped = true; }
          forced = prev_rejected && p.h_min > 0.0 && h == p.h_min;
          ys = fma(h_try * dp::a21, k1, y);
          ts = fma(dp::c2, h_try, t);
          break;
        case 2: ys = fma(h_try, fma(dp::a32, k2, dp::a31 * k1), y); ts = fma(dp::c3, h_try, t); break;
        case 3:
          ys = fma(h_try, fma(dp::a43, k3, fma(dp::a42, k2, dp::a41 * k1)), y);
          ts = fma(dp::c4, h_try, t);
          break;
        case 4:
          ys = fma(h_try, fma(dp::a54, k4, fma(dp::a53, k3, fma(dp::a52, k2, dp::a51 * k1))), y);
          ts = fma(dp::c5, h_try, t);
          break;
        case 5:
          ys = fma(h_try, fma(dp::a65, k5, fma(dp::a64, k4, fma(dp::a63, k3, fma(dp::a62, k2, dp::a61 * k1)))), y);
          ts = t + h_try;
          break;
        default:
          yn = fma(h_try, fma(dp::a76, k6, fma(dp::a75, k5, fma(dp::a74, k4, fma(dp::a73, k3, dp::a71 * k1)))), y);
          ys = yn;
          ts = t + h_try;
          break;
      }
      if (stage == 1 && !(t + h_try > t)) { st = GC_ST_NONFINITE_; break; }     // step underflow
      double kv;
      {
        const double s_ = shfl_d(ys, 0), th_ = shfl_d(ys, 1), ze_ = shfl_d(ys, 2), u_ = shfl_d(ys, 3);
        double dy[4];
        rhs(f, sc, role, lane, p.mass, p.charge, mu, p.v_ref, p.inv_v_ref, ts, s_, th_, ze_, u_, dy);
        kv = comp == 0 ? dy[0] : comp == 1 ? dy[1] : comp == 2 ? dy[2] : dy[3];
      }
      switch (stage) {
        case 0: k1 = kv; break;
        case 1: k2 = kv; break;
        case 2: k3 = kv; break;
        case 3: k4 = kv; break;
        case 4: k5 = kv; break;
        case 5: k6 = kv; break;
        default: k7 = kv; break;
      }
      if (stage == 0) {
        if (!__all_sync(kFull, isfinite(y) && isfinite(k1))) st = GC_ST_NONFINITE_;   // O6: checked before the
        else if (!(t < p.t_max)) st = 0;                                              // t0 >= t_max shortcut
        stage = 1;
        continue;
      }
      if (stage < 6) { ++stage; continue; }
      stage = 1;

      // ---- a7: error norm and controller (O6) --------------------------------------------------------------
      ++attempts;
      const double delta = h_try * fma(dp::e7, k7, fma(dp::e6, k6, fma(dp::e5, k5, fma(dp::e4, k4,
                                   fma(dp::e3, k3, dp::e1 * k1)))));
      const double sk = fma(p.rtol, fmax(fabs(y), fabs(yn)), p.atol);
      const double r = delta / sk;
      // sum of the four components in index order 0..3, the same on every lane
      const double r0 = shfl_d(r, 0), r1 = shfl_d(r, 1), r2 = shfl_d(r, 2), r3 = shfl_d(r, 3);
      const double err = sqrt(fma(r3, r3, fma(r2, r2, fma(r1, r1, r0 * r0))) * 0.25);
      const bool finite = __all_sync(kFull, isfinite(yn) && isfinite(k7)) && isfinite(err);
      bool accept;
      if (forced) {
        if (!finite) { st = GC_ST_NONFINITE_; break; }
        accept = true;
      } else {
        accept = finite && err <= 1.0;
      }
      if (accept) {
        const double scl = scale_after_accept(err);
        const double h_next = prev_rejected ? h_try * fmin(scl, 1.0) : h_try * scl;
        if (p.poincare_capacity > 0) {
          const double z0 = shfl_d(y, 2), z1 = shfl_d(yn, 2);
          if (floor(z0 / kTwoPi) != floor(z1 / kTwoPi)) {
            const double q2 = yn - y;
            const double q3 = h_try * k1 - q2;
            const double q4 = q2 - h_try * k7 - q3;
            const double q5 = h_try * fma(dp::d7, k7, fma(dp::d6, k6, fma(dp::d5, k5, fma(dp::d4, k4,
                                      fma(dp::d3, k3, dp::d1 * k1)))));
            Dense3 d;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
              d.r1[c] = shfl_d(y, c); d.r2[c] = shfl_d(q2, c); d.r3[c] = shfl_d(q3, c);
              d.r4[c] = shfl_d(q4, c); d.r5[c] = shfl_d(q5, c);
            }
            if (lane == 0) poincare_emit(d, i, t, h_try, z0, z1, p.poincare, p.poincare_capacity, p.poincare_count);
            __syncwarp();
          }
        }
        t = clipped ? p.t_max : t + h_try;
        y = yn;
        k1 = k7;
        ++n_acc;
        if (forced) ++n_forced;
        prev_rejected = false;
        if (!clipped) h = h_next;
        if (h < p.h_min) h = p.h_min;
        const double s_now = shfl_d(y, 0);
        if (s_now >= p.s_loss) st = 1;
        else if (s_now <= p.s_min) st = 2;
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
    // a8: result store, lanes 0..3 write the four components
    if (lane < 4) p.y_out[(long long)comp * p.n + i] = comp == 3 ? y * p.v_ref : y;
    if (lane == 0) {
      p.t_out[i] = t;
      p.status[i] = st;
      if (p.h_inout) p.h_inout[i] = h;
      // counters restart at 0 per call, except under GC_TRACE_RESUME where they add to what is there
      if (p.n_acc) p.n_acc[i] = (p.resume ? p.n_acc[i] : 0) + n_acc;
      if (p.n_rej) p.n_rej[i] = (p.resume ? p.n_rej[i] : 0) + n_rej;
      if (p.n_forced) p.n_forced[i] = (p.resume ? p.n_forced[i] : 0) + n_forced;
    }
  }
}

// One warp per state: the warp kernel's right-hand side alone (gc_rhs_eval, parity tests of O4).
template <int NIT_MAIN, int NX, bool MODES, int NREG>
__global__ void __launch_bounds__(kWarpsPerBlock * 32, 1)
rhs_eval_warp_kernel(FieldDev f, double mass, double charge, double t, long long n, const double* y,
                     const double* mu, double* dydt) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  WarpScratch& sc = reinterpret_cast<WarpScratch*>(gc_dyn_smem)[warp];
  init_scratch(sc, lane);
  const LaneRole role = make_role(f, lane);
  WarpRhs<NIT_MAIN, NX, MODES, NREG> rhs;
  rhs.win.sm = warp_window_smem<NIT_MAIN, NX, MODES, NREG>(warp, lane);
  rhs.cur_i0 = -1000;
  rhs.inv_mass = 1.0 / mass;
  rhs.inv_charge = 1.0 / charge;
  for (long long i = (long long)blockIdx.x * kWarpsPerBlock + warp; i < n;
       i += (long long)gridDim.x * kWarpsPerBlock) {
    double dy[4];
    rhs(f, sc, role, lane, mass, charge, mu[i], 1.0, 1.0, t, y[i], y[n + i], y[2 * n + i], y[3 * n + i], dy);
    if (lane < 4) dydt[(long long)lane * n + i] = lane == 0 ? dy[0] : lane == 1 ? dy[1] : lane == 2 ? dy[2] : dy[3];
  }
}

}  // namespace gc
