// fast3d.cuh -- fused H psi / ABM stage kernels for 3-D lattices with Ny = Nz = 32 (Nx in {8, 16, 32}), the
// regime of configs[3] (32^3): every lattice line is transformed in the registers of ONE thread (regfft.cuh),
// planes are transposed once through padded shared memory, and the 3-D transform is split into
//   pass A  x-planes : load psi (coalesced, lane = z), FFT y, transpose, FFT z        -> spec  [c][x][kz][ky]
//   pass B  x-lines  : FFT x, times -k^2 / M (Eq. 26), inverse FFT x, in place, no shared memory
//   pass C  x-planes : inverse FFT z, transpose, inverse FFT y, then the pointwise BdG mix (Eqs. 5, 15, 40),
//                      eps_n partial sums (Eq. 44b) and the ABM combination of the stage (Alg. 2), all in registers.
// The spectra live in chunk-sized scratch that stays in the 126 MB L2; HBM sees psi in, result out.
// Kinetic forms: LAPLACE (Eq. 14) and SYM40 (Eq. 40); DIVGRAD stays on the general path.
#pragma once
#include "regfft.cuh"

#define F3_N 32                    // Ny = Nz
#define F3_PITCH 33                // padded row of the transposition tile (conflict-free 16-byte column reads)
#define F3_PLANE (F3_N * F3_N)
#define F3_TILE_BYTES (F3_N * F3_PITCH * 16)

struct F3Fields {
  const double *alpha[2], *lap[2], *U[2];
  const cplx *delta, *dext;
  double mu[2];
};

// fixed-order warp sum (shuffle tree); every lane gets the result
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---- pass A -------------------------------------------------------------------------------------------------
struct F3PassA {
  const cplx* psi;            // chunk base, [cnt][2][NX][32][32]
  const double* scale;        // per spinor of the chunk (nullable): psi is used as scale_n * psi
  const double* alpha[2];     // SYM: second spectrum is that of alpha_c * w
  cplx* spec0;                // [cnt * 2][NX][kz][ky]
  cplx* spec1;
  int n_items;                // cnt * 2 * NX   (one warp per component plane)
  int NX;
};

// forward 2-D transform of the plane held one line per lane (x[j] = (j, lane)): FFT along j, transpose through
// the padded tile, FFT along the other axis; returns x[j] = (k_other = j, k_first = lane).  The loop is NOT
// unrolled so that the 32-point butterfly code exists once (instruction-cache footprint).
__device__ __forceinline__ void f3_plane_forward(cplx* x, cplx* S, int lane) {
#pragma unroll 1
  for (int pass = 0; pass < 2; ++pass) {
    fft_reg<F3_N, false>(x);
    if (pass == 0) {
#pragma unroll
      for (int j = 0; j < F3_N; ++j) S[j * F3_PITCH + lane] = x[j];
      __syncwarp();
#pragma unroll
      for (int j = 0; j < F3_N; ++j) x[j] = S[lane * F3_PITCH + j];
      __syncwarp();
    }
  }
}

template <bool SYM>
__global__ void __launch_bounds__(128, 3) k_f3_pass_a(F3PassA a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  cplx* S = reinterpret_cast<cplx*>(smem_raw) + warp * (F3_N * F3_PITCH);
  cplx x[F3_N];
  for (int item = blockIdx.x * 4 + warp; item < a.n_items; item += gridDim.x * 4) {
    const int ix = item % a.NX, cc = item / a.NX, c = cc & 1;
    const double s = a.scale ? a.scale[cc >> 1] : 1.0;
    const cplx* src = a.psi + (size_t)item * F3_PLANE;
    const double* al = a.alpha[c] + (size_t)ix * F3_PLANE;
#pragma unroll 1
    for (int t = 0; t < (SYM ? 2 : 1); ++t) {
#pragma unroll
      for (int j = 0; j < F3_N; ++j) {
        double f = s;
        if (SYM && t) f *= al[j * F3_N + lane];
        x[j] = cscale(src[j * F3_N + lane], f);                  // (y = j, z = lane)
      }
      f3_plane_forward(x, S, lane);                              // (kz = j, ky = lane)
      cplx* dst = (t == 0 ? a.spec0 : a.spec1) + (size_t)item * F3_PLANE;
#pragma unroll
      for (int j = 0; j < F3_N; ++j) dst[j * F3_N + lane] = x[j];
    }
  }
}

// ---- pass B -------------------------------------------------------------------------------------------------
struct F3PassB {
  cplx* spec[2];
  int n_spec;                 // 1 or 2
  int n_items;                // cnt * 2 * 32  (one warp per (component, kz); lane = ky)
  const double* ky2;          // k_y^2, k_z^2 in natural index order (Eq. 25), Nyquist kept
  const double* kz2;
  double kx2[32];             // k_x^2, natural order
  double invM;
};

// The inverse transform is conj(FFT(conj(x))) (exact: conjugation only flips signs), so only the forward
// butterfly code is instantiated and the two directions share one loop body.
template <int NX>
__global__ void __launch_bounds__(128, 3) k_f3_pass_b(F3PassB a) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  cplx x[NX];
  for (int item = blockIdx.x * 4 + warp; item < a.n_items; item += gridDim.x * 4) {
    const int kz = item & (F3_N - 1), cc = item >> 5;
    const double kyz2 = a.ky2[lane] + a.kz2[kz];
#pragma unroll 1
    for (int t = 0; t < a.n_spec; ++t) {
      cplx* p = a.spec[t] + (size_t)cc * NX * F3_PLANE + kz * F3_N + lane;
#pragma unroll
      for (int j = 0; j < NX; ++j) x[j] = p[(size_t)j * F3_PLANE];
#pragma unroll 1
      for (int dir = 0; dir < 2; ++dir) {
        fft_reg<NX, false>(x);
#pragma unroll
        for (int j = 0; j < NX; ++j) {
          const double f = dir ? 1.0 : -(a.kx2[j] + kyz2) * a.invM;     // even derivative: Nyquist kept
          x[j] = make_double2(x[j].x * f, -x[j].y * f);                 // conj(x) * f
        }
      }
#pragma unroll
      for (int j = 0; j < NX; ++j) p[(size_t)j * F3_PLANE] = x[j];
    }
  }
}

// ---- pass C -------------------------------------------------------------------------------------------------
enum { F3_APPLY = 0, F3_CORR = 1, F3_RHS = 2 };
#define F3_NPART 5            // per (spinor, x-plane) partial sums: e, |X|^2, Re/Im sum conj(X) w, |w|^2

struct F3PassC {
  const cplx* spec0;          // lap w spectra after pass B, [cnt * 2][NX][kz][ky]
  const cplx* spec1;          // SYM: lap(alpha w)
  const cplx* psi;            // chunk base
  const double* scale;        // nullable
  const double* kperp2;       // per spinor of the chunk
  F3Fields F;
  cplx* out;                  // APPLY: H psi;  CORR: X = C_part - i kappa H psi;  RHS: Y = -i H psi   [cnt][2][M]
  const cplx* cpart;          // CORR
  double kappa;               // CORR: c_0 dt
  double* part;               // [F3_NPART][cnt * NX]
  int n_items;                // cnt * NX   (one warp per (spinor, x-plane), both components)
  int NX;
};

template <bool SYM, int MODE>
__global__ void __launch_bounds__(64, SYM ? 3 : 6) k_f3_pass_c(F3PassC a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  constexpr int PER_WARP = F3_N * F3_PITCH + (SYM ? F3_PLANE : 0);
  cplx* S = reinterpret_cast<cplx*>(smem_raw) + warp * PER_WARP;
  cplx* T = S + F3_N * F3_PITCH;                               // SYM: alpha * lap w, thread-private slots
  const size_t M = (size_t)a.NX * F3_PLANE;
  const int np = a.n_items;
  cplx x[F3_N];
  for (int item = blockIdx.x * 2 + warp; item < a.n_items; item += gridDim.x * 2) {
    const int ix = item % a.NX, n = item / a.NX;
    const double s = a.scale ? a.scale[n] : 1.0, kp2 = a.kperp2[n];
    const size_t pl = (size_t)ix * F3_PLANE;                    // plane offset inside a field / component
    const cplx* pu = a.psi + (size_t)(2 * n) * M + pl;
    const cplx* pv = pu + M;
    double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
#pragma unroll 1
    for (int c = 0; c < 2; ++c) {
      const size_t cplane = ((size_t)(2 * n + c) * a.NX + ix) * F3_PLANE;
      const double* al = a.F.alpha[c] + pl;
#pragma unroll 1
      for (int t = 0; t < (SYM ? 2 : 1); ++t) {
        const cplx* sp = (t ? a.spec1 : a.spec0) + cplane;
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = cconj(sp[j * F3_N + lane]);        // (kz = j, ky = lane), conjugated
        f3_plane_forward(x, S, lane);                                             // conj of value at (y = j, z = lane)
        if (SYM && t == 0) {
#pragma unroll
          for (int j = 0; j < F3_N; ++j) T[j * F3_N + lane] = cscale(cconj(x[j]), al[j * F3_N + lane]);
        } else {
#pragma unroll
          for (int j = 0; j < F3_N; ++j) S[j * F3_PITCH + lane] = cconj(x[j]);   // own column: thread-private
        }
      }
      const double* lp = a.F.lap[c] + pl;
      const double* Uc = a.F.U[c] + pl;
      const double mu = a.F.mu[c];
      const size_t ob = (size_t)(2 * n + c) * M + pl;
#pragma unroll 4
      for (int j = 0; j < F3_N; ++j) {
        const int i = j * F3_N + lane;
        const cplx u = cscale(pu[i], s), v = cscale(pv[i], s);
        const cplx w = c ? v : u;
        const cplx L = S[j * F3_PITCH + lane];
        cplx K;
        if (SYM) {
          const cplx t = T[i];
          const double a_ = al[i], l_ = lp[i], h = 0.5 * a_ * kp2;
          K.x = -0.25 * (L.x + t.x - l_ * w.x) + h * w.x;        // Eq. 40 + transverse shift
          K.y = -0.25 * (L.y + t.y - l_ * w.y) + h * w.y;
        } else {
          K.x = -0.5 * L.x + 0.5 * kp2 * w.x;                    // Eq. 14
          K.y = -0.5 * L.y + 0.5 * kp2 * w.y;
        }
        const cplx D = cadd(a.F.delta[pl + i], a.F.dext[pl + i]);
        const double pot = Uc[i] - mu;
        cplx H;
        if (c == 0) H = cadd(K, cadd(cscale(u, pot), cmul(D, v)));                // Eqs. 5, 15
        else H = csub(cmul(cconj(D), u), cadd(K, cscale(v, pot)));
        e += w.x * H.x + w.y * H.y;
        cplx o;
        if (MODE == F3_APPLY) o = H;
        else if (MODE == F3_RHS) o = make_double2(H.y, -H.x);                      // -i H
        else {
          const cplx cp = a.cpart[ob + i];
          o = make_double2(cp.x + a.kappa * H.y, cp.y - a.kappa * H.x);           // C_part - i kappa H
          xx += cabs2(o); xpr += o.x * w.x + o.y * w.y; xpi += o.x * w.y - o.y * w.x; pp += cabs2(w);
        }
        a.out[ob + i] = o;
      }
    }
    e = warp_sum(e);
    if (MODE == F3_CORR) { xx = warp_sum(xx); xpr = warp_sum(xpr); xpi = warp_sum(xpi); pp = warp_sum(pp); }
    if (lane == 0) {
      a.part[item] = e;
      if (MODE == F3_CORR) { a.part[np + item] = xx; a.part[2 * np + item] = xpr; a.part[3 * np + item] = xpi; a.part[4 * np + item] = pp; }
    }
  }
}

// ---- per-spinor scalars from the pass-C partial sums (one warp per spinor, fixed summation order) ---------------
struct F3Scal {
  const double* part;         // [F3_NPART][cnt * NX]
  int cnt, NX, mode, use_shift, normalize;
  double dV, kappa;
  double* eps;                // out, per spinor of the chunk: eps_n = Re dV sum psi^+ H psi (Eq. 44b), 0 when the shift is off
  double* eps_user;           // nullable second copy (wslda_apply_h's eps_dev): always the true eps_n
  double* scale_new;          // CORR: 1 / sqrt(dV sum |phi_new|^2) (Alg. 2 step 8), or 1
};

__global__ void k_f3_scal(F3Scal a) {
  const int n = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (n >= a.cnt) return;
  const int np = a.cnt * a.NX;
  double v[F3_NPART];
#pragma unroll
  for (int k = 0; k < F3_NPART; ++k) {
    double t = 0.0;
    if ((k == 0 || a.mode == F3_CORR) && lane < a.NX) t = a.part[k * np + n * a.NX + lane];
    v[k] = warp_sum(t);
  }
  if (lane) return;
  const double e_true = a.dV * v[0], e = a.use_shift ? e_true : 0.0;
  a.eps[n] = e;
  if (a.eps_user) a.eps_user[n] = e_true;
  if (a.mode == F3_CORR) {
    // |X + i kappa eps w|^2 summed = xx - 2 kappa eps Im(xp) + kappa^2 eps^2 pp
    const double ke = a.kappa * e, nrm2 = a.dV * (v[1] - 2.0 * ke * v[3] + ke * ke * v[4]);
    a.scale_new[n] = a.normalize ? 1.0 / sqrt(nrm2) : 1.0;
  }
}

// ---- stage epilogues ----------------------------------------------------------------------------------------
struct F3Dens {                // density accumulation of a chunk into a per-stream accumulator [4][M]
  const double *cpref, *w_a, *w_b;     // per spinor of the chunk
  double* acc;                 // planes rho_a, rho_b, nu_re, nu_im (Eqs. 7a, 7b, 7e)
  int first;                   // 1: overwrite, 0: add
};

// Alg. 2 step 4 + 8: phi_new = (X + i kappa eps w) * scale_new, w = scale_P * P, written over P;
// optionally the densities of phi_new.  One thread per lattice point, spinors of the chunk in increasing n.
struct F3Fin2 {
  const cplx* X;
  cplx* phi;
  const double *scaleP, *eps, *scale_new;
  double kappa;
  int cnt;
  int64_t M;
  int do_dens;
  F3Dens d;
};

__device__ __forceinline__ void f3_dens_add(double* acc4, cplx u, cplx v, double cp, double wa, double wb) {
  acc4[0] += cp * wa * cabs2(u);
  acc4[1] += cp * wb * cabs2(v);
  const double wn = 0.5 * cp * (wb - wa);
  acc4[2] += wn * (u.x * v.x + u.y * v.y);
  acc4[3] += wn * (u.y * v.x - u.x * v.y);
}
__device__ __forceinline__ void f3_dens_store(const F3Dens& d, int64_t M, int64_t i, const double* acc4) {
#pragma unroll
  for (int f = 0; f < 4; ++f) d.acc[f * M + i] = (d.first ? 0.0 : d.acc[f * M + i]) + acc4[f];
}

__global__ void __launch_bounds__(128) k_f3_fin2(F3Fin2 a) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.M) return;
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll 2
  for (int n = 0; n < a.cnt; ++n) {
    const double sP = a.scaleP ? a.scaleP[n] : 1.0, ke = a.kappa * a.eps[n], sn = a.scale_new[n];
    const int64_t ou = (int64_t)(2 * n) * a.M + i, ov = ou + a.M;
    const cplx xu = a.X[ou], xv = a.X[ov];
    const cplx wu = cscale(a.phi[ou], sP), wv = cscale(a.phi[ov], sP);
    const cplx u = make_double2((xu.x - ke * wu.y) * sn, (xu.y + ke * wu.x) * sn);
    const cplx v = make_double2((xv.x - ke * wv.y) * sn, (xv.y + ke * wv.x) * sn);
    a.phi[ou] = u; a.phi[ov] = v;
    if (a.do_dens) f3_dens_add(acc, u, v, a.d.cpref[n], a.d.w_a[n], a.d.w_b[n]);
  }
  if (a.do_dens) f3_dens_store(a.d, a.M, i, acc);
}

// densities of scale_n * psi for the spinors of a chunk (stage 1: the normalised predictor)
struct F3DensOnly { const cplx* psi; const double* scale; int cnt; int64_t M; F3Dens d; };
// 64 lattice points per CTA, the chunk's spinors dealt round-robin to four thread groups (more loads in flight: the kernel
// is bound by L2 latency, not by arithmetic); the four partial sums are added in a fixed order
__global__ void __launch_bounds__(256) k_f3_dens(F3DensOnly a) {
  __shared__ double part[3][4][64];
  const int p = threadIdx.x & 63, q = threadIdx.x >> 6;
  const int64_t i = (int64_t)blockIdx.x * 64 + p;                 // M is a multiple of 1024 on this path
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll 4
  for (int n = q; n < a.cnt; n += 4) {
    const double s = a.scale ? a.scale[n] : 1.0;
    const cplx u = cscale(a.psi[(int64_t)(2 * n) * a.M + i], s), v = cscale(a.psi[(int64_t)(2 * n + 1) * a.M + i], s);
    f3_dens_add(acc, u, v, a.d.cpref[n], a.d.w_a[n], a.d.w_b[n]);
  }
  if (q) {
#pragma unroll
    for (int f = 0; f < 4; ++f) part[q - 1][f][p] = acc[f];
  }
  __syncthreads();
  if (q == 0) {
#pragma unroll
    for (int f = 0; f < 4; ++f) acc[f] = (acc[f] + part[0][f][p]) + (part[1][f][p] + part[2][f][p]);
    f3_dens_store(a.d, a.M, i, acc);
  }
}

// raw[f] = sum over the per-stream accumulators in stream order (planes rho_a, rho_b, nu_re, nu_im)
__global__ void k_f3_dens_final(const double* acc, int n_streams, int64_t stride, int64_t M, double* raw) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= 4 * M) return;
  double s = 0.0;
  for (int k = 0; k < n_streams; ++k) s += acc[k * stride + i];
  raw[i] = s;
}

// Alg. 2 step 9: f = Y + i eps phi  (Y = -i H phi from pass C; Eq. 45b)
__global__ void __launch_bounds__(256) k_f3_fin3(const cplx* Y, const cplx* phi, const double* eps, cplx* f, int64_t M2) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y;
  if (i >= M2) return;
  const double e = eps[n];
  const int64_t o = n * M2 + i;
  const cplx y = Y[o], p = phi[o];
  f[o] = make_double2(y.x - e * p.y, y.y + e * p.x);
}
