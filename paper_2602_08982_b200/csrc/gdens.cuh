// gdens.cuh -- the gradient densities tau_sigma and j_sigma (Eqs. 7c-d, 7f-g PAPER.md:164-178) on cubic 3-D lattices
// (32^3, 64^3: configs[3], configs[4]) without ever materialising a gradient.
//
// |grad w|^2 = sum_d |d_d w|^2 and j_d need d_d w only, and the spectral derivative along axis d (Eq. 26 PAPER.md:369,
// odd derivative: Nyquist mode dropped) is a 1-D transform pair on every line of that axis.  So each axis
// is an independent pass: a thread (32-point lines) or a pair of threads (64-point lines, mega64.cuh) holds one line in
// registers, takes d_d w with two register transforms, and adds c_n w_n |d_d w|^2 and -/+ c_n w_n Im[w d_d w^*] for its
// points into thread-private shared-memory accumulators while it loops over the spinors of its group (increasing n:
// fixed order).  HBM sees psi three times (once per axis) instead of one forward and three inverse 3-D transforms
// through scratch (general path: 82 us per spinor at 64^3).  Grid: (line tiles, 3 axes x 2 spins, spinor groups);
// partial planes part[g][d][sigma][tau | j_d][M] are summed in index order by k_gdens_reduce (bit-reproducible).
#pragma once
#include "mega64.cuh"

struct GdArgs {
  const cplx* psi;              // first spinor of the range, [n][2][M]
  const double *cpref, *w_a, *w_b;   // per spinor of the range
  const double* scale;          // per spinor, nullable: the densities of scale_n psi_n (the unnormalised predictor)
  double kd[3][64];             // wave numbers of Eq. 25, natural order, Nyquist entry zeroed (odd derivative)
  double* part;                 // [G][3][2][2][M]
  int n, G;                     // spinors in the range, groups
};

template <int N> struct GdLine;
template <> struct GdLine<32> {
  static constexpr int LINES = 128;                               // per 128-thread CTA
  int q;
  __device__ __forceinline__ GdLine() : q(threadIdx.x) {}
  __device__ __forceinline__ int idx(int j) const { return j; }
  // x <- conj(d w / d line) at the points idx(j); in: x[j] = w at idx(j)
  __device__ __forceinline__ void deriv(cplx* x, const double* k) const {
    fft_reg<32, false>(x);
#pragma unroll
    for (int j = 0; j < 32; ++j) { const double f = k[j] * (1.0 / 32.0); x[j] = make_double2(-f * x[j].y, -f * x[j].x); }   // conj(i k X / N)
    fft_reg<32, false>(x);
  }
  // x <- conj(d^2 w / d line^2); k2: squared wave numbers, natural order, Nyquist mode kept (even derivative)
  __device__ __forceinline__ void deriv2(cplx* x, const double* k2) const {
    fft_reg<32, false>(x);
#pragma unroll
    for (int j = 0; j < 32; ++j) { const double f = -k2[j] * (1.0 / 32.0); x[j] = make_double2(f * x[j].x, -f * x[j].y); }       // conj(-k^2 X / N)
    fft_reg<32, false>(x);
  }
};
template <> struct GdLine<64> {
  static constexpr int LINES = 64;
  int q, p;
  __device__ __forceinline__ GdLine() { const int lane = threadIdx.x & 31; p = lane >> 4; q = (threadIdx.x >> 5) * 16 + (lane & 15); }
  __device__ __forceinline__ int idx(int j) const { return 2 * j + p; }
  __device__ __forceinline__ void deriv(cplx* x, const double* k) const {
    f6_dit(x, p);                                                 // block spectrum: x[j] = X[j + 32 p]
#pragma unroll
    for (int j = 0; j < 32; ++j) { const double f = k[j + 32 * p] * (1.0 / 64.0); x[j] = make_double2(-f * x[j].y, -f * x[j].x); }
    f6_dif(x, p);                                                 // interleaved again: conj of the derivative at 2 j + p
  }
  __device__ __forceinline__ void deriv2(cplx* x, const double* k2) const {
    f6_dit(x, p);
#pragma unroll
    for (int j = 0; j < 32; ++j) { const double f = -k2[j + 32 * p] * (1.0 / 64.0); x[j] = make_double2(f * x[j].x, -f * x[j].y); }
    f6_dif(x, p);
  }
};

// WHAT: bit 0 = tau, bit 1 = j (a step that consumes only one of them skips the other's accumulators and, for tau alone, the
// second read of the line)
template <int N, int WHAT = 3>
__global__ void __launch_bounds__(128, 2) k_gdens(const __grid_constant__ GdArgs a) {
  extern __shared__ double gd_acc[];                              // [2][32][128]: tau, j_d of this thread's 32 points
  const GdLine<N> L;
  const int d = blockIdx.y >> 1, sg = blockIdx.y & 1, g = blockIdx.z;
  const int line = blockIdx.x * GdLine<N>::LINES + L.q;           // in [0, N * N): the two coordinates other than d
  const int c0 = line / N, c1 = line - c0 * N;
  const size_t M = (size_t)N * N * N;
  size_t base, stride;
  if (d == 0) { base = (size_t)c0 * N + c1; stride = (size_t)N * N; }            // (y, z) fixed, x runs
  else if (d == 1) { base = (size_t)c0 * N * N + c1; stride = N; }               // (x, z) fixed, y runs
  else { base = ((size_t)c0 * N + c1) * N; stride = 1; }                         // (x, y) fixed, z runs
  double* aT = gd_acc + threadIdx.x;
  double* aJ = aT + 32 * 128;
#pragma unroll
  for (int j = 0; j < 32; ++j) { if (WHAT & 1) aT[j * 128] = 0.0; if (WHAT & 2) aJ[j * 128] = 0.0; }
  const int per = (a.n + a.G - 1) / a.G, n0 = g * per, n1 = min(a.n, n0 + per);
  const double* wt = sg ? a.w_b : a.w_a;
  const double sgn = sg ? 1.0 : -1.0;                             // Eq. 7f: j_a = -sum Im[u grad u^*]; Eq. 7g: j_b = +sum Im[v grad v^*]
  cplx x[32];
#pragma unroll 1
  for (int n = n0; n < n1; ++n) {
    const double sc = a.scale ? a.scale[n] : 1.0, cw = a.cpref[n] * wt[n] * (sc * sc);
    if (cw == 0.0) continue;                                      // uniform over the CTA (e.g. w_a = 0 with Eq. 8 weights)
    const cplx* src = a.psi + (size_t)(2 * n + sg) * M + base;
#pragma unroll
    for (int j = 0; j < 32; ++j) x[j] = src[(size_t)L.idx(j) * stride];
    L.deriv(x, a.kd[d]);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      if (WHAT & 1) aT[j * 128] += cw * (x[j].x * x[j].x + x[j].y * x[j].y);
      if (WHAT & 2) {
        const cplx w = src[(size_t)L.idx(j) * stride];            // again (L1 / L2): the line registers held the transform
        aJ[j * 128] += sgn * cw * (w.y * x[j].x + w.x * x[j].y);  // Im[w conj(d w)] with x = conj(d w)
      }
    }
  }
  double* pT = a.part + ((((size_t)g * 3 + d) * 2 + sg) * 2) * M + base;
  double* pJ = pT + M;
#pragma unroll
  for (int j = 0; j < 32; ++j) {
    if (WHAT & 1) pT[(size_t)L.idx(j) * stride] = aT[j * 128];
    if (WHAT & 2) pJ[(size_t)L.idx(j) * stride] = aJ[j * 128];
  }
}

// raw tau_sigma = sum_g sum_d part, raw j_sigma,d = sum_g part (index order); mask selects TAU / J planes
__global__ void k_gdens_reduce(const double* part, int G, int64_t M, double* raw, unsigned mask, int accumulate) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
#pragma unroll
  for (int sg = 0; sg < 2; ++sg) {
    double t = 0.0, j[3] = {0.0, 0.0, 0.0};
    for (int g = 0; g < G; ++g)
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const double* p = part + ((((int64_t)g * 3 + d) * 2 + sg) * 2) * M + i;
        t += p[0]; j[d] += p[M];
      }
    if (mask & WSLDA_D_TAU) { double* r = raw + (int64_t)(DP_TAU_A + sg) * M + i; *r = (accumulate ? *r : 0.0) + t; }
    if (mask & WSLDA_D_J)
#pragma unroll
      for (int d = 0; d < 3; ++d) { double* r = raw + (int64_t)((sg ? DP_JB0 : DP_JA0) + d) * M + i; *r = (accumulate ? *r : 0.0) + j[d]; }
  }
}

// ---- the kinetic anomalous density B' = -1/2 sum_n wn [u lap v^* + v^* lap u] (Eq. 68; weights of nu, R29) the same
// way: lap = sum of the second derivatives along the axes, each a pass over the lines of one axis.  The thread holding a line of u
// adds v^* d_d^2 u, the one holding a line of v adds u (d_d^2 v)^* (the other component is read at the line's points); partial
// planes [G][3][2][re | im][M] as above, summed in index order by k_gdens_bp_reduce.  a.kd holds the SQUARED wave numbers here.
template <int N>
__global__ void __launch_bounds__(128, 2) k_gdens_bp(const __grid_constant__ GdArgs a) {
  extern __shared__ double gd_acc[];
  const GdLine<N> L;
  const int d = blockIdx.y >> 1, sg = blockIdx.y & 1, g = blockIdx.z;
  const int line = blockIdx.x * GdLine<N>::LINES + L.q;
  const int c0 = line / N, c1 = line - c0 * N;
  const size_t M = (size_t)N * N * N;
  size_t base, stride;
  if (d == 0) { base = (size_t)c0 * N + c1; stride = (size_t)N * N; }
  else if (d == 1) { base = (size_t)c0 * N * N + c1; stride = N; }
  else { base = ((size_t)c0 * N + c1) * N; stride = 1; }
  double* aR = gd_acc + threadIdx.x;
  double* aI = aR + 32 * 128;
#pragma unroll
  for (int j = 0; j < 32; ++j) { aR[j * 128] = 0.0; aI[j * 128] = 0.0; }
  const int per = (a.n + a.G - 1) / a.G, n0 = g * per, n1 = min(a.n, n0 + per);
  cplx x[32];
#pragma unroll 1
  for (int n = n0; n < n1; ++n) {
    const double sc = a.scale ? a.scale[n] : 1.0, wn = -0.25 * a.cpref[n] * (a.w_b[n] - a.w_a[n]) * (sc * sc);   // -1/2 x 1/2 c_n (w_b - w_a)
    if (wn == 0.0) continue;
    const cplx* src = a.psi + (size_t)(2 * n + sg) * M + base;
    const cplx* oth = a.psi + (size_t)(2 * n + 1 - sg) * M + base;
#pragma unroll
    for (int j = 0; j < 32; ++j) x[j] = src[(size_t)L.idx(j) * stride];
    L.deriv2(x, a.kd[d]);                                         // x = conj(d_d^2 w)
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      const cplx o = oth[(size_t)L.idx(j) * stride];
      // sg = 0: v^* d^2 u = conj(v x);  sg = 1: u (d^2 v)^* = u x
      const double re = o.x * x[j].x - o.y * x[j].y, im = o.x * x[j].y + o.y * x[j].x;
      aR[j * 128] += wn * re;
      aI[j * 128] += (sg ? wn : -wn) * im;
    }
  }
  double* pR = a.part + ((((size_t)g * 3 + d) * 2 + sg) * 2) * M + base;
  double* pI = pR + M;
#pragma unroll
  for (int j = 0; j < 32; ++j) { pR[(size_t)L.idx(j) * stride] = aR[j * 128]; pI[(size_t)L.idx(j) * stride] = aI[j * 128]; }
}

__global__ void k_gdens_bp_reduce(const double* part, int G, int64_t M, double* raw, int accumulate) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  double re = 0.0, im = 0.0;
  for (int g = 0; g < G; ++g)
#pragma unroll
    for (int d = 0; d < 3; ++d)
#pragma unroll
      for (int sg = 0; sg < 2; ++sg) {
        const double* p = part + ((((int64_t)g * 3 + d) * 2 + sg) * 2) * M + i;
        re += p[0]; im += p[M];
      }
  double* r = raw + (int64_t)DP_BP_RE * M + i;
  r[0] = (accumulate ? r[0] : 0.0) + re;
  r[M] = (accumulate ? r[M] : 0.0) + im;
}
