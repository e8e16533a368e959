// common.cuh -- types shared by the kernels of libwslda (CUDA, sm_100a).  Not part of the C-ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/wslda.h"

typedef double2 cplx;

#define WS_MAX_SCR 8          // chunk-sized scratch buffers carved from the workspace
#define WS_PT_THREADS 256     // threads of the pointwise kernels
#define WS_NFIELD_D 11        // raw density planes: rho_a rho_b tau_a tau_b nu_re nu_im is packed separately

__host__ __device__ inline cplx cmul(cplx a, cplx b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__host__ __device__ inline cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__host__ __device__ inline cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__host__ __device__ inline cplx cscale(cplx a, double s) { return make_double2(a.x * s, a.y * s); }
__host__ __device__ inline cplx cconj(cplx a) { return make_double2(a.x, -a.y); }
__host__ __device__ inline double cabs2(cplx a) { return a.x * a.x + a.y * a.y; }

// Lattice + transform tables, passed by value to kernels.
struct Lat {
  int nd;               // held axes
  int N[3];             // sizes of the held axes (1 for non-held)
  int lg[3];            // log2 N
  int64_t M;            // points per component
  const cplx* tw[3];    // tw[d][j] = exp(-2 pi i j / N_d), j < N_d
  const double* kk[3];  // wave number (Eq. 25) at STORED position p of the in-place transform, Nyquist kept
  const double* ko[3];  // same with the Nyquist entry zeroed (odd derivatives)
  double invM;
};

// One batched derivative request: for components c_local in [0, ncomp):
//   w = src[(src_comp0 + c_local) * M + i] * scale[(src_comp0 + c_local) / 2] * premul[(src_comp0 + c_local) & 1][i]
//   out[0] = lap w, out[1+j] = d_j w   (null = not wanted), each laid out [c_local][M].
struct DerivArgs {
  const cplx* src;
  int64_t src_comp0;
  int ncomp;
  const double* scale;
  const double* premul[2];
  cplx* out[4];
};

// deterministic block sum (fixed order: lanes by shuffle tree, then warps in index order); result in thread 0
__device__ inline double block_sum(double v, double* sh /* >= 32 doubles */) {
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (l == 0) sh[w] = v;
  __syncthreads();
  double r = 0.0;
  if (threadIdx.x == 0) for (int i = 0; i < nw; ++i) r += sh[i];
  return r;
}
