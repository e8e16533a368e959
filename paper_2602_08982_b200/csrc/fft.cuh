// fft.cuh -- batched complex128 FFTs in shared memory and the spectral-derivative kernels (Eqs. 25-26,
// PAPER.md:360-371).  Forward = decimation in frequency, in place, natural order in -> digit-reversed
// order out; inverse = the exact transpose (decimation in time), digit-reversed in -> natural out.  The
// k-space multiply runs on the digit-reversed data with k-tables stored in that order, so no reordering
// pass and no second buffer are needed.  Radix 8 (register butterflies) with a final radix-4 / radix-2 stage.
#pragma once
#include "common.cuh"
#include "regfft.cuh"

// One axis of a block laid out [A][n][B] (element (a,j,b) at (a*n + j)*B + b) in shared memory.
// All sizes are powers of two; lgn = log2 n, lgB = log2 B.  tw[j] = exp(-2 pi i j / n).
// Radix plan: 8 while the remaining length is >= 8, then the remainder (4 or 2): 8 -> one pass, 64 -> two, 128 -> three.
// Each thread pulls the R strided points of a butterfly into registers, runs the unrolled register transform of
// regfft.cuh, applies the twiddles and writes back in place -- R-fold fewer shared-memory passes and barriers than
// radix-2, and the butterfly arithmetic runs out of registers with full ILP.
template <bool INV, int R>
__device__ inline void fft_stage(cplx* s, int A, int lgn, int lgL, int lgB, const cplx* __restrict__ tw) {
  constexpr int lgR = R == 8 ? 3 : R == 4 ? 2 : 1;
  const int lgq = lgL - lgR, items = A << (lgn - lgR + lgB), Bm = (1 << lgB) - 1;
  for (int t = threadIdx.x; t < items; t += blockDim.x) {
    const int b = t & Bm, r = t >> lgB;
    const int qq = r & ((1 << (lgn - lgR)) - 1), a = r >> (lgn - lgR);
    const int q = qq & ((1 << lgq) - 1), blk = qq >> lgq;
    cplx* p = s + ((((size_t)a << lgn) + ((size_t)blk << lgL) + q) << lgB) + b;
    const size_t st = (size_t)1 << (lgq + lgB);
    const int e = q << (lgn - lgL);                            // W_L^q = tw[q * n / L]
    cplx x[R];
#pragma unroll
    for (int m = 0; m < R; ++m) x[m] = p[m * st];
    if (!INV) {                                                // DIF: butterfly, then twiddle W_L^(q m)
      fft_reg<R, false>(x);
      if (q) {
#pragma unroll
        for (int m = 1; m < R; ++m) x[m] = cmul(x[m], __ldg(tw + m * e));
      }
    } else {                                                   // DIT: conj twiddle, then the inverse butterfly
      if (q) {
#pragma unroll
        for (int m = 1; m < R; ++m) x[m] = cmul(x[m], cconj(__ldg(tw + m * e)));
      }
#pragma unroll
      for (int m = 0; m < R; ++m) x[m] = cconj(x[m]);          // inverse = conj(forward(conj))
      fft_reg<R, false>(x);
#pragma unroll
      for (int m = 0; m < R; ++m) x[m] = cconj(x[m]);
    }
#pragma unroll
    for (int m = 0; m < R; ++m) p[m * st] = x[m];
  }
  __syncthreads();
}

// largest radix of the plan (log2): 3 = radix 8, 2 = radix 4; set once per process from WSLDA_FFT_RADIX (ctx.cuh keeps
// the permuted k-tables consistent with it)
__device__ int g_ws_lgr = 3;

template <bool INV>
__device__ inline void fft_axis(cplx* s, int A, int lgn, int lgB, const cplx* __restrict__ tw) {
  if (lgn == 0) return;
  const int lgr = g_ws_lgr, rem = lgn % lgr;                   // last (smallest) stage: radix 2^rem
  if (!INV) {
    for (int lgL = lgn; lgL >= lgr; lgL -= lgr) {
      if (lgr == 3) fft_stage<false, 8>(s, A, lgn, lgL, lgB, tw); else fft_stage<false, 4>(s, A, lgn, lgL, lgB, tw);
    }
    if (rem == 2) fft_stage<false, 4>(s, A, lgn, 2, lgB, tw);
    else if (rem == 1) fft_stage<false, 2>(s, A, lgn, 1, lgB, tw);
  } else {
    if (rem == 2) fft_stage<true, 4>(s, A, lgn, 2, lgB, tw);
    else if (rem == 1) fft_stage<true, 2>(s, A, lgn, 1, lgB, tw);
    for (int lgL = rem + lgr; lgL <= lgn; lgL += lgr) {
      if (lgr == 3) fft_stage<true, 8>(s, A, lgn, lgL, lgB, tw); else fft_stage<true, 4>(s, A, lgn, lgL, lgB, tw);
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
