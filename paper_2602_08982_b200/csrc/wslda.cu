// wslda.cu -- the single translation unit of libwslda (C-ABI in include/wslda.h).
// Build: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -lineinfo -shared -Xcompiler -fPIC wslda.cu -o libwslda.so
#include "step.cuh"

// ---------------------------------------------------------------------------------------------------------------------
// wslda_gradient_densities_static -- the gradient densities tau_sigma, j_sigma (Eqs. 7c-d, 7f-g PAPER.md:164-178) of a
// batch of spinors on a cubic 32^3 or 64^3 lattice, for callers that cannot allocate (CUDA graph capture, serving
// loops): no context, no workspace, no cudaMalloc.  It is the axis-by-axis kernel of gdens.cuh with its partial planes
// [group][axis][spin][tau | j_d][M] in a file-scope device array instead of the caller's workspace.  Every GPU that
// loads the library holds the array (24 MiB) until exit; every call shares it, so calls that overlap on the GPU race.
// Nothing in it has to start at zero: a call overwrites every partial plane it later reads.
#include <mutex>
#define WS_STATIC_SCRATCH_BYTES (24u << 20)               // 8 groups x 12 planes at 32^3, 1 group x 12 planes at 64^3
static __device__ __align__(256) unsigned char g_static_scratch[WS_STATIC_SCRATCH_BYTES];

struct GsArgs {
  const cplx* psi;              // [n][2][M]
  const double *cw_a, *cw_b;    // per spinor: c_n w^a_n, c_n w^b_n (prefactor of Eqs. 29-30 times the weight of Eqs. 7 / 8)
  double kd[3][64];             // wave numbers of Eq. 25, natural order, Nyquist entry zeroed (odd derivative)
  double* part;                 // the static scratch, [G][3][2][2][M]
  int n, G;
};

// the variant of k_gdens (gdens.cuh): same lines, same order of summation (increasing n inside a group)
template <int N>
__global__ void __launch_bounds__(128, 2) k_gdens_static(const __grid_constant__ GsArgs a) {
  extern __shared__ double gs_acc[];                              // [2][32][128]
  const GdLine<N> L;
  const int d = blockIdx.y >> 1, sg = blockIdx.y & 1, g = blockIdx.z;
  const int line = blockIdx.x * GdLine<N>::LINES + L.q;
  const int c0 = line / N, c1 = line - c0 * N;
  const size_t M = (size_t)N * N * N;
  size_t base, stride;
  if (d == 0) { base = (size_t)c0 * N + c1; stride = (size_t)N * N; }
  else if (d == 1) { base = (size_t)c0 * N * N + c1; stride = N; }
  else { base = ((size_t)c0 * N + c1) * N; stride = 1; }
  double* aT = gs_acc + threadIdx.x;
  double* aJ = aT + 32 * 128;
#pragma unroll
  for (int j = 0; j < 32; ++j) { aT[j * 128] = 0.0; aJ[j * 128] = 0.0; }
  const int per = (a.n + a.G - 1) / a.G, n0 = g * per, n1 = min(a.n, n0 + per);
  const double* wt = sg ? a.cw_b : a.cw_a;
  const double sgn = sg ? 1.0 : -1.0;                             // Eqs. 7f, 7g
  cplx x[32];
#pragma unroll 1
  for (int n = n0; n < n1; ++n) {
    const double cw = wt[n];
    if (cw == 0.0) continue;
    const cplx* src = a.psi + (size_t)(2 * n + sg) * M + base;
#pragma unroll
    for (int j = 0; j < 32; ++j) x[j] = src[(size_t)L.idx(j) * stride];
    L.deriv(x, a.kd[d]);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      const cplx w = src[(size_t)L.idx(j) * stride];
      aT[j * 128] += cw * (x[j].x * x[j].x + x[j].y * x[j].y);
      aJ[j * 128] += sgn * cw * (w.y * x[j].x + w.x * x[j].y);
    }
  }
  double* pT = a.part + ((((size_t)g * 3 + d) * 2 + sg) * 2) * M + base;
  double* pJ = pT + M;
#pragma unroll
  for (int j = 0; j < 32; ++j) { pT[(size_t)L.idx(j) * stride] = aT[j * 128]; pJ[(size_t)L.idx(j) * stride] = aJ[j * 128]; }
}

// tau[sg][M] = sum_g sum_d part, j[sg][d][M] = sum_g part (index order: bit-reproducible)
__global__ void k_gdens_static_reduce(const double* part, int G, int64_t M, double* tau, double* j) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
#pragma unroll
  for (int sg = 0; sg < 2; ++sg) {
    double t = 0.0, jj[3] = {0.0, 0.0, 0.0};
    for (int g = 0; g < G; ++g)
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const double* p = part + ((((int64_t)g * 3 + d) * 2 + sg) * 2) * M + i;
        t += p[0]; jj[d] += p[M];
      }
    if (tau) tau[(int64_t)sg * M + i] = t;
    if (j)
#pragma unroll
      for (int d = 0; d < 3; ++d) j[((int64_t)sg * 3 + d) * M + i] = jj[d];
  }
}

// once per device, with that device current: the device address of the scratch (the name g_static_scratch is only a
// host-side stand-in in host code) and the kernels' dynamic shared-memory limit.  Neither call allocates.
#define WS_STATIC_MAX_DEVICES 64
static std::mutex g_static_mu;
static double* g_static_ptr[WS_STATIC_MAX_DEVICES];
static bool g_static_ready[WS_STATIC_MAX_DEVICES];
static wslda_status static_setup(int dev, double** ptr) {
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ready[dev]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_gdens_static<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_gdens_static<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      snprintf(g_err, 256, "gradient_densities_static: set-up failed on device %d: %s", dev, cudaGetErrorString(e));
      return WSLDA_ECUDA;
    }
    g_static_ptr[dev] = (double*)p;
    g_static_ready[dev] = true;
  }
  *ptr = g_static_ptr[dev];
  return WSLDA_OK;
}

extern "C" size_t wslda_static_scratch_bytes(void) { return WS_STATIC_SCRATCH_BYTES; }

extern "C" wslda_status wslda_gradient_densities_static(const void* psi, const double* cw_a, const double* cw_b, int64_t n_wf,
                                                        int n_side, const double dx[3], double* tau, double* j, void* stream) {
  if (!psi || !cw_a || !cw_b || !dx || (!tau && !j)) return fail(nullptr, WSLDA_EINVAL, "gradient_densities_static: null argument");
  if (n_side > WSLDA_STATIC_MAX_SIDE) {
    snprintf(g_err, 256, "gradient_densities_static: lattice side %d is beyond the maximum of %d (the static scratch holds 12 planes of %d^3 doubles)",
             n_side, WSLDA_STATIC_MAX_SIDE, WSLDA_STATIC_MAX_SIDE);
    return WSLDA_EINVAL;
  }
  if (n_side != 32 && n_side != 64) return fail(nullptr, WSLDA_EINVAL, "gradient_densities_static: the lattice must be cubic with side 32 or 64");
  if (n_wf < 1 || n_wf > WSLDA_STATIC_MAX_SPINORS) {
    snprintf(g_err, 256, "gradient_densities_static: %lld spinors, must be in [1, %d]", (long long)n_wf, WSLDA_STATIC_MAX_SPINORS);
    return WSLDA_EINVAL;
  }
  if (!(dx[0] > 0.0) || !(dx[1] > 0.0) || !(dx[2] > 0.0)) return fail(nullptr, WSLDA_EINVAL, "gradient_densities_static: dx must be positive");
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= WS_STATIC_MAX_DEVICES) {
    cudaGetLastError();
    return fail(nullptr, WSLDA_ECUDA, "gradient_densities_static: no current CUDA device (or a device ordinal beyond 63)");
  }
  GsArgs a;
  wslda_status rc = static_setup(dev, &a.part);
  if (rc != WSLDA_OK) return rc;
  const int N = n_side;
  const int64_t M = (int64_t)N * N * N;
  a.psi = (const cplx*)psi; a.cw_a = cw_a; a.cw_b = cw_b; a.n = (int)n_wf;
  const double PI = 3.14159265358979323846264338327950288;
  for (int d = 0; d < 3; ++d) {
    const double len = N * dx[d];
    for (int q = 0; q < 64; ++q) a.kd[d][q] = (q >= N || q == N / 2) ? 0.0 : (q < N / 2 ? 2.0 * PI * q / len : 2.0 * PI * (q - N) / len);
  }
  int G = (int)(WS_STATIC_SCRATCH_BYTES / (12 * M * 8));        // 8 at 32^3, 1 at 64^3
  if (G > n_wf) G = (int)n_wf;
  a.G = G;
  cudaStream_t st = (cudaStream_t)stream;
  const int tiles = N * N / (N == 32 ? 128 : 64);
  if (N == 32) k_gdens_static<32><<<dim3(tiles, 6, G), 128, 2 * 32 * 128 * 8, st>>>(a);
  else k_gdens_static<64><<<dim3(tiles, 6, G), 128, 2 * 32 * 128 * 8, st>>>(a);
  k_gdens_static_reduce<<<(unsigned)((M + 255) / 256), 256, 0, st>>>(a.part, G, M, tau, j);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { snprintf(g_err, 256, "gradient_densities_static: launch failed: %s", cudaGetErrorString(e)); return WSLDA_ECUDA; }
  return WSLDA_OK;
}
