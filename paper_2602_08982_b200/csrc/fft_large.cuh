// fft_large.cuh -- spectral derivatives of lattices too large for one CTA's shared memory (32^3, 64^3, ...).
// The component [Nx][R] (R = Ny*Nz in 3D, Ny in 2D) takes three passes whose intermediates live in
// chunk-sized scratch that stays in the 126 MB L2:
//   A  x-planes: load, scale/premultiply, forward FFT over the R axes            -> spec   [c][Nx][R]
//   B  x-lines : forward x, k-multiply per output, inverse x                     -> out[o] [c][Nx][R]
//   C  x-planes: inverse FFT over the R axes, in place in out[o]
#pragma once
#include "fft.cuh"

// grid (Nx / PX, ncomp); smem PX * R * 16
__global__ void __launch_bounds__(256) k_planes_fwd(Lat L, DerivArgs a, cplx* spec, int PX) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* F = reinterpret_cast<cplx*>(smem_raw);
  const int lgR = L.lg[1] + L.lg[2];
  const int64_t M = L.M;
  const int c = blockIdx.y, x0 = blockIdx.x * PX, tot = PX << lgR;
  const int64_t base = (int64_t)x0 << lgR;
  for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) F[idx] = load_src(a, c, M, base + idx);
  __syncthreads();
  if (L.nd > 2) fft_axis<false>(F, PX << L.lg[1], L.lg[2], 0, L.tw[2]);
  fft_axis<false>(F, PX, L.lg[1], L.lg[2], L.tw[1]);
  cplx* dst = spec + (int64_t)c * M + base;
  for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) dst[idx] = F[idx];
}

// grid (R / T, ncomp); smem 2 * Nx * T * 16
__global__ void __launch_bounds__(256) k_xlines(Lat L, const cplx* __restrict__ spec, DerivArgs a, int lgT) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* F = reinterpret_cast<cplx*>(smem_raw);
  const int lgR = L.lg[1] + L.lg[2], T = 1 << lgT;
  const int64_t M = L.M;
  const int c = blockIdx.y, r0 = blockIdx.x << lgT, tot = L.N[0] << lgT;
  cplx* W = F + tot;
  const cplx* src = spec + (int64_t)c * M + r0;
  for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) {
    int x = idx >> lgT, b = idx & (T - 1);
    F[idx] = src[((int64_t)x << lgR) + b];
  }
  __syncthreads();
  fft_axis<false>(F, 1, L.lg[0], lgT, L.tw[0]);
  for (int o = 0; o < 4; ++o) {
    if (!a.out[o]) continue;
    for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) {
      int x = idx >> lgT, r = r0 + (idx & (T - 1));
      int j2 = r & (L.N[2] - 1), j1 = r >> L.lg[2];
      W[idx] = cmul(F[idx], kfactor(L, o, x, j1, j2));
    }
    __syncthreads();
    fft_axis<true>(W, 1, L.lg[0], lgT, L.tw[0]);
    cplx* dst = a.out[o] + (int64_t)c * M + r0;
    for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) {
      int x = idx >> lgT, b = idx & (T - 1);
      dst[((int64_t)x << lgR) + b] = W[idx];
    }
    __syncthreads();
  }
}

// grid (Nx / PX, ncomp, n_out); outs[blockIdx.z] is transformed in place
struct OutList { cplx* p[4]; };
__global__ void __launch_bounds__(256) k_planes_inv(Lat L, OutList outs, int PX) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* F = reinterpret_cast<cplx*>(smem_raw);
  const int lgR = L.lg[1] + L.lg[2];
  const int c = blockIdx.y, x0 = blockIdx.x * PX, tot = PX << lgR;
  cplx* buf = outs.p[blockIdx.z] + (int64_t)c * L.M + ((int64_t)x0 << lgR);
  for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) F[idx] = buf[idx];
  __syncthreads();
  fft_axis<true>(F, PX, L.lg[1], L.lg[2], L.tw[1]);
  if (L.nd > 2) fft_axis<true>(F, PX << L.lg[1], L.lg[2], 0, L.tw[2]);
  for (int idx = threadIdx.x; idx < tot; idx += blockDim.x) buf[idx] = F[idx];
}
