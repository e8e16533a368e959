// fft.cuh -- batched complex128 FFTs in shared memory and the spectral-derivative kernels (Eqs. 25-26,
// PAPER.md:360-371).  Forward = decimation in frequency, in place, natural order in -> digit-reversed
// order out; inverse = the exact transpose (decimation in time), digit-reversed in -> natural out.  The
// k-space multiply runs on the digit-reversed data with k-tables stored in that order, so no reordering
// pass and no second buffer are needed.  Radix 4 with a final radix-2 stage when log2 N is odd.
#pragma once
#include "common.cuh"

// One axis of a block laid out [A][n][B] (element (a,j,b) at (a*n + j)*B + b) in shared memory.
// All sizes are powers of two; lgn = log2 n, lgB = log2 B.  tw[j] = exp(-2 pi i j / n).
template <bool INV>
__device__ inline void fft_axis(cplx* s, int A, int lgn, int lgB, const cplx* __restrict__ tw) {
  const int n = 1 << lgn;
  if (n == 1) return;
  const int Bm = (1 << lgB) - 1;
  const bool odd = lgn & 1;
  if (!INV) {
    for (int lgL = lgn; lgL >= 2; lgL -= 2) {                 // radix-4 DIF stages, L = n, n/4, ...
      const int lgq = lgL - 2, items = A << (lgn - 2 + lgB);
      for (int t = threadIdx.x; t < items; t += blockDim.x) {
        int b = t & Bm, r = t >> lgB;
        int qq = r & ((n >> 2) - 1), a = r >> (lgn - 2);
        int q = qq & ((1 << lgq) - 1), blk = qq >> lgq;
        cplx* p = s + ((((size_t)a << lgn) + ((size_t)blk << lgL) + q) << lgB) + b;
        const size_t st = (size_t)1 << (lgq + lgB);
        cplx a0 = p[0], a1 = p[st], a2 = p[2 * st], a3 = p[3 * st];
        cplx b0 = cadd(a0, a2), b1 = csub(a0, a2), b2 = cadd(a1, a3), d = csub(a1, a3);
        cplx b3 = make_double2(d.y, -d.x);                    // (a1 - a3) * (-i)
        cplx y0 = cadd(b0, b2), y1 = cadd(b1, b3), y2 = csub(b0, b2), y3 = csub(b1, b3);
        if (q) {
          int e = q << (lgn - lgL);                           // W_L^q = tw[q * n / L]
          y1 = cmul(y1, tw[e]); y2 = cmul(y2, tw[2 * e]); y3 = cmul(y3, tw[3 * e]);
        }
        p[0] = y0; p[st] = y1; p[2 * st] = y2; p[3 * st] = y3;
      }
      __syncthreads();
    }
    if (odd) {                                                // final radix-2 stage, L = 2, no twiddle
      const int items = A << (lgn - 1 + lgB);
      for (int t = threadIdx.x; t < items; t += blockDim.x) {
        int b = t & Bm, r = t >> lgB;
        cplx* p = s + ((size_t)(2 * r) << lgB) + b;
        cplx a0 = p[0], a1 = p[(size_t)1 << lgB];
        p[0] = cadd(a0, a1); p[(size_t)1 << lgB] = csub(a0, a1);
      }
      __syncthreads();
    }
  } else {
    if (odd) {
      const int items = A << (lgn - 1 + lgB);
      for (int t = threadIdx.x; t < items; t += blockDim.x) {
        int b = t & Bm, r = t >> lgB;
        cplx* p = s + ((size_t)(2 * r) << lgB) + b;
        cplx a0 = p[0], a1 = p[(size_t)1 << lgB];
        p[0] = cadd(a0, a1); p[(size_t)1 << lgB] = csub(a0, a1);
      }
      __syncthreads();
    }
    for (int lgL = odd ? 3 : 2; lgL <= lgn; lgL += 2) {       // radix-4 DIT stages, L = 4 (8), ..., n
      const int lgq = lgL - 2, items = A << (lgn - 2 + lgB);
      for (int t = threadIdx.x; t < items; t += blockDim.x) {
        int b = t & Bm, r = t >> lgB;
        int qq = r & ((n >> 2) - 1), a = r >> (lgn - 2);
        int q = qq & ((1 << lgq) - 1), blk = qq >> lgq;
        cplx* p = s + ((((size_t)a << lgn) + ((size_t)blk << lgL) + q) << lgB) + b;
        const size_t st = (size_t)1 << (lgq + lgB);
        cplx y0 = p[0], y1 = p[st], y2 = p[2 * st], y3 = p[3 * st];
        if (q) {
          int e = q << (lgn - lgL);
          y1 = cmul(y1, cconj(tw[e])); y2 = cmul(y2, cconj(tw[2 * e])); y3 = cmul(y3, cconj(tw[3 * e]));
        }
        cplx b0 = cadd(y0, y2), b1 = csub(y0, y2), b2 = cadd(y1, y3), d = csub(y1, y3);
        cplx b3 = make_double2(-d.y, d.x);                    // (y1 - y3) * (+i)
        p[0] = cadd(b0, b2); p[st] = cadd(b1, b3); p[2 * st] = csub(b0, b2); p[3 * st] = csub(b1, b3);
      }
      __syncthreads();
    }
  }
}

// k-space factor of output o (0: Laplacian -k^2, 1+j: i k_j with the axis-j Nyquist mode zeroed) at the
// stored position (j0, j1, j2); the 1/M of the inverse transform (Eq. 26) is folded in.
__device__ inline cplx kfactor(const Lat& L, int o, int j0, int j1, int j2) {
  if (o == 0) {
    double k2 = L.kk[0][j0] * L.kk[0][j0];
    if (L.nd > 1) k2 += L.kk[1][j1] * L.kk[1][j1];
    if (L.nd > 2) k2 += L.kk[2][j2] * L.kk[2][j2];
    return make_double2(-k2 * L.invM, 0.0);
  }
  int ax = o - 1;
  double k = L.ko[ax][ax == 0 ? j0 : (ax == 1 ? j1 : j2)];
  return make_double2(0.0, k * L.invM);
}

__device__ inline cplx load_src(const DerivArgs& a, int c_local, int64_t M, int64_t i) {
  int64_t cg = a.src_comp0 + c_local;
  cplx v = a.src[cg * M + i];
  double f = 1.0;
  if (a.scale) f = a.scale[cg >> 1];
  const double* pm = a.premul[cg & 1];
  if (pm) f *= pm[i];
  return (a.scale || pm) ? cscale(v, f) : v;
}

// Whole lattice of G components per CTA in shared memory: forward over all held axes, then one inverse per
// requested output.  Dynamic smem = 2 * G * M * 16 bytes (F and W).
__global__ void __launch_bounds__(256) k_deriv_onchip(Lat L, DerivArgs a, int G) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* F = reinterpret_cast<cplx*>(smem_raw);
  const int64_t M = L.M;
  const int tot = (int)(G * M);
  cplx* W = F + tot;
  const int c0 = blockIdx.x * G;
  for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) {
    int g = idx / (int)M, i = idx - g * (int)M;
    F[idx] = (c0 + g < a.ncomp) ? load_src(a, c0 + g, M, i) : make_double2(0.0, 0.0);
  }
  __syncthreads();
  const int lgM = L.lg[0] + L.lg[1] + L.lg[2];
  // axis d of block [G * prod_{e<d} N_e][N_d][prod_{e>d} N_e]
  if (L.nd > 2) fft_axis<false>(F, G << (L.lg[0] + L.lg[1]), L.lg[2], 0, L.tw[2]);
  if (L.nd > 1) fft_axis<false>(F, G << L.lg[0], L.lg[1], L.lg[2], L.tw[1]);
  fft_axis<false>(F, G, L.lg[0], L.lg[1] + L.lg[2], L.tw[0]);
  for (int o = 0; o < 4; ++o) {
    if (!a.out[o]) continue;
    for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) {
      int i = idx & ((1 << lgM) - 1);
      int j2 = i & (L.N[2] - 1), j1 = (i >> L.lg[2]) & (L.N[1] - 1), j0 = i >> (L.lg[1] + L.lg[2]);
      W[idx] = cmul(F[idx], kfactor(L, o, j0, j1, j2));
    }
    __syncthreads();
    fft_axis<true>(W, G, L.lg[0], L.lg[1] + L.lg[2], L.tw[0]);
    if (L.nd > 1) fft_axis<true>(W, G << L.lg[0], L.lg[1], L.lg[2], L.tw[1]);
    if (L.nd > 2) fft_axis<true>(W, G << (L.lg[0] + L.lg[1]), L.lg[2], 0, L.tw[2]);
    for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) {
      int g = idx / (int)M, i = idx - g * (int)M;
      if (c0 + g < a.ncomp) a.out[o][(int64_t)(c0 + g) * M + i] = W[idx];
    }
    __syncthreads();
  }
}
