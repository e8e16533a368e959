// kernels.cuh -- pointwise and reduction kernels of the TDSLDA step (general, unfused path).
// Grids are (blocks over the M lattice points, spinors of the chunk); per-spinor arrays and spinor
// buffers are passed already offset to the first spinor of the chunk.
#pragma once
#include "common.cuh"

struct HistPtrs { const cplx* f[5]; };
struct AbmCoef { double b[5]; double c[5]; int ab, am; };   // b_i * dt, c_i * dt (c[0] multiplies f(P))

// Alg. 2 step 1: P = phi + dt sum b_i f_i -> phi buffer; C_part = phi + dt sum_{i>=1} c_i f_i
// -> oldest history buffer; per-block partial sums of |P|^2 (Alg. 2 step 2 needs the norm).
__global__ void __launch_bounds__(WS_PT_THREADS) k_abm_combine(cplx* phi, HistPtrs h, cplx* cpart, AbmCoef k, int64_t M,
                                                               double* part, int nblk) {
  __shared__ double sh[32];
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y;
  double acc = 0.0;
  if (i < M) {
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const int64_t o = (2 * n + c) * M + i;
      cplx p = phi[o], q = p;
#pragma unroll
      for (int j = 0; j < 5; ++j) {
        if (j < k.ab || j + 1 < k.am) {
          cplx f = h.f[j][o];
          if (j < k.ab) { p.x += k.b[j] * f.x; p.y += k.b[j] * f.y; }
          if (j + 1 < k.am) { q.x += k.c[j + 1] * f.x; q.y += k.c[j + 1] * f.y; }
        }
      }
      phi[o] = p; cpart[o] = q;
      acc += cabs2(p);
    }
  }
  if (part) { double r = block_sum(acc, sh); if (threadIdx.x == 0) part[n * nblk + blockIdx.x] = r; }
}

// per-block partial sums of |psi|^2 only (norm of an existing buffer)
// The same predictor sweep for the fused 3-D path (chunks of a few dozen MB on concurrent streams): the history and
// phi are read for the last time in this stage (L2 evict_first), C_part is not needed before the next stage
// (evict_first), while P is re-read by the density kernel of the same chunk and must stay in L2 (evict_last).
// The CTA that completes a spinor's partial sums (a self-resetting arrival counter per spinor) turns them into
// scale_n = 1 / sqrt(dV sum |P|^2) in the fixed order of k_from_partials: no separate launch per chunk.
__global__ void __launch_bounds__(WS_PT_THREADS) k_f3_combine(cplx* phi, HistPtrs h, cplx* cpart, AbmCoef k, int64_t M,
                                                              double* part, int nblk, int* arrived, double dV, double* scale) {
  __shared__ double sh[32];
  __shared__ int s_last;
  const F3Pol pol = f3_policies();
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y;
  double acc = 0.0;
  if (i < M) {
    cplx p0[2], fh[2][5];
#pragma unroll
    for (int c = 0; c < 2; ++c) {                               // all loads of the point first
      const int64_t o = (2 * n + c) * M + i;
      p0[c] = ld_pol(phi + o, pol.drop);
#pragma unroll
      for (int j = 0; j < 5; ++j)
        if (j < k.ab || j + 1 < k.am) fh[c][j] = ld_pol(h.f[j] + o, pol.drop);
    }
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const int64_t o = (2 * n + c) * M + i;
      cplx p = p0[c], q = p;
#pragma unroll
      for (int j = 0; j < 5; ++j) {
        if (j < k.ab) { p.x += k.b[j] * fh[c][j].x; p.y += k.b[j] * fh[c][j].y; }
        if (j + 1 < k.am) { q.x += k.c[j + 1] * fh[c][j].x; q.y += k.c[j + 1] * fh[c][j].y; }
      }
      st_pol_nb(phi + o, p, pol.keep); st_pol_nb(cpart + o, q, pol.drop);
      acc += cabs2(p);
    }
  }
  if (!part) return;
  const double r = block_sum(acc, sh);
  if (threadIdx.x == 0) {
    part[n * nblk + blockIdx.x] = r;
    __threadfence();
    s_last = atomicAdd(arrived + n, 1) == nblk - 1;
  }
  __syncthreads();
  if (!s_last || threadIdx.x >= 32) return;
  __threadfence();
  double s = 0.0;
  for (int b = threadIdx.x; b < nblk; b += 32) s += __ldcg(part + n * nblk + b);
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (threadIdx.x == 0) { scale[n] = 1.0 / sqrt(s * dV); arrived[n] = 0; }
}

__global__ void __launch_bounds__(WS_PT_THREADS) k_norm_partials(const cplx* psi, int64_t M, double* part, int nblk) {
  __shared__ double sh[32];
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y;
  double acc = 0.0;
  if (i < M) acc = cabs2(psi[2 * n * M + i]) + cabs2(psi[(2 * n + 1) * M + i]);
  double r = block_sum(acc, sh);
  if (threadIdx.x == 0) part[n * nblk + blockIdx.x] = r;
}

// scale_n = 1 / sqrt(dV * sum_blk part) (Eq. 16 with n = m), or eps_n = dV * sum_blk part (Eq. 44b)
__global__ void k_from_partials(const double* part, int nblk, int64_t n_count, double dV, int as_scale, double* out,
                                double* out2) {
  // one warp per spinor: lanes take the partials in stride-32 order, then a fixed shuffle tree (deterministic)
  const int64_t n = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (n >= n_count) return;
  double s = 0.0;
  for (int b = lane; b < nblk; b += 32) s += part[n * nblk + b];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane) return;
  double r = as_scale ? 1.0 / sqrt(s * dV) : s * dV;
  out[n] = r;
  if (out2) out2[n] = r;
}

__global__ void k_fill(double* p, int64_t n, double v) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

// in-place psi_n *= scale_n
__global__ void __launch_bounds__(WS_PT_THREADS) k_scale_spinors(cplx* psi, const double* scale, int64_t M) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y;
  if (i >= M) return;
  const double s = scale[n];
  cplx* p = psi + 2 * n * M;
  p[i] = cscale(p[i], s); p[M + i] = cscale(p[M + i], s);
}

struct Fields {
  const double *alpha_a, *alpha_b, *lap_a, *lap_b, *U_a, *U_b;
  const cplx *delta, *dext;
  double mu_a, mu_b;
};

// Pointwise BdG mix (Eqs. 5, 15 PAPER.md:154, 289) from the spectral terms held in scratch s0..s2, laid out
// [2 n + c][M]:  LAPLACE s0 = lap w;  SYM40 s0 = lap w, s1 = lap(alpha w);  DIVGRAD s_j = d_j(alpha d_j w).
// psi is scaled by scale_n on the fly.  Writes H psi and per-block partial sums of Re psi^+ H psi.
// cur (nullable): {W_sigma, grad} w of the current / velocity coupling, same layout; it enters both rows as -(i/2) cur
// (Eq. 4c; the v row holds -h_b^*, whose coupling term is -conj(-(i/2){W, grad}) = -(i/2){W, grad}).
__global__ void __launch_bounds__(WS_PT_THREADS) k_hmix(const cplx* psi, const double* scale, const double* kperp2,
                                                        int kin, int nd, const cplx* s0, const cplx* s1, const cplx* s2,
                                                        Fields F, int64_t M, cplx* out, double* epart, int nblk, const cplx* cur) {
  __shared__ double sh[32];
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y;
  double acc = 0.0;
  if (i < M) {
    const double s = scale ? scale[n] : 1.0, kp2 = kperp2[n];
    const int64_t ou = 2 * n * M + i, ov = ou + M;
    const cplx u = cscale(psi[ou], s), v = cscale(psi[ov], s);
    cplx K[2];
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const int64_t o = c ? ov : ou;
      const cplx w = c ? v : u;
      const double al = c ? F.alpha_b[i] : F.alpha_a[i];
      cplx r;
      if (kin == WSLDA_KIN_LAPLACE) {
        cplx l = s0[o];
        r = make_double2(-0.5 * l.x + 0.5 * kp2 * w.x, -0.5 * l.y + 0.5 * kp2 * w.y);
      } else if (kin == WSLDA_KIN_SYM40) {
        cplx l = s0[o], la = s1[o];
        const double lp = c ? F.lap_b[i] : F.lap_a[i];
        r.x = -0.25 * (la.x + al * l.x - lp * w.x) + 0.5 * al * kp2 * w.x;
        r.y = -0.25 * (la.y + al * l.y - lp * w.y) + 0.5 * al * kp2 * w.y;
      } else {
        cplx d = s0[o];
        if (nd > 1) d = cadd(d, s1[o]);
        if (nd > 2) d = cadd(d, s2[o]);
        r.x = -0.5 * d.x + 0.5 * al * kp2 * w.x;
        r.y = -0.5 * d.y + 0.5 * al * kp2 * w.y;
      }
      K[c] = r;
    }
    const cplx D = cadd(F.delta[i], F.dext[i]);
    const double pa = F.U_a[i] - F.mu_a, pb = F.U_b[i] - F.mu_b;
    cplx hu = cadd(K[0], cadd(cscale(u, pa), cmul(D, v)));
    cplx hv = csub(cmul(cconj(D), u), cadd(K[1], cscale(v, pb)));
    if (cur) {
      const cplx cu = cur[ou], cv = cur[ov];
      hu.x += 0.5 * cu.y; hu.y -= 0.5 * cu.x;
      hv.x += 0.5 * cv.y; hv.y -= 0.5 * cv.x;
    }
    out[ou] = hu; out[ov] = hv;
    acc = u.x * hu.x + u.y * hu.y + v.x * hv.x + v.y * hv.y;   // Re(conj(u) hu + conj(v) hv)
  }
  if (epart) { double r = block_sum(acc, sh); if (threadIdx.x == 0) epart[n * nblk + blockIdx.x] = r; }
}

// Right-hand side f = -i (H psi - eps psi) (Eq. 45b) and what follows it.
//  mode 0: dst = f; if write_back, src <- psi (the normalised state)
//  mode 1: src <- C_part + cdt * f  (Alg. 2 step 4), per-block partial sums of its |.|^2
__global__ void __launch_bounds__(WS_PT_THREADS) k_rhs(cplx* src, const double* scale, const cplx* hpsi, const double* eps,
                                                       int mode, int write_back, cplx* dst, const cplx* cpart, double cdt,
                                                       int64_t M, double* part, int nblk) {
  __shared__ double sh[32];
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y;
  double acc = 0.0;
  if (i < M) {
    const double s = scale ? scale[n] : 1.0, e = eps ? eps[n] : 0.0;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const int64_t o = (2 * n + c) * M + i;
      const cplx w = cscale(src[o], s), h = hpsi[o];
      const cplx g = make_double2(h.x - e * w.x, h.y - e * w.y);
      const cplx f = make_double2(g.y, -g.x);                 // -i g
      if (mode == 0) {
        dst[o] = f;
        if (write_back) src[o] = w;
      } else {
        cplx q = cpart[o];
        q.x += cdt * f.x; q.y += cdt * f.y;
        src[o] = q;
        acc += cabs2(q);
      }
    }
  }
  if (part) { double r = block_sum(acc, sh); if (threadIdx.x == 0) part[n * nblk + blockIdx.x] = r; }
}

// Taylor starter accumulation (Eqs. 53-54): g = H t - eps t; t <- g; out += coef * g
__global__ void __launch_bounds__(WS_PT_THREADS) k_taylor_acc(cplx* t, const cplx* ht, const double* eps, cplx coef, cplx* out,
                                                              int64_t M) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, n = blockIdx.y;
  if (i >= M) return;
  const double e = eps ? eps[n] : 0.0;
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    const int64_t o = (2 * n + c) * M + i;
    cplx tt = t[o], h = ht[o];
    cplx g = make_double2(h.x - e * tt.x, h.y - e * tt.y);
    t[o] = g;
    out[o] = cadd(out[o], cmul(coef, g));
  }
}

__global__ void k_copy2(const cplx* src, cplx* a, cplx* b, int64_t n) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) { cplx v = src[i]; a[i] = v; if (b) b[i] = v; }
}
__global__ void k_real_to_cplx(const double* a, const double* b, cplx* dst, int64_t M) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < M) { dst[i] = make_double2(a[i], 0.0); dst[M + i] = make_double2(b[i], 0.0); }
}
__global__ void k_cplx_real_part(const cplx* src, double* a, double* b, int64_t M) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < M) { a[i] = src[i].x; b[i] = src[M + i].x; }
}

// current / velocity coupling, accumulation of {W, grad} w = sum_d [ W_d (d_d w) + d_d (W_d w) ]:
//   acc (=, +=) f[sigma of the component][i] * t   (f = W_d, [2][M] with stride 3 M between the spins; null: factor 1)
__global__ void k_cur_acc(cplx* acc, const cplx* t, const double* f, int64_t fstride, int64_t M, int64_t ncomp, int first) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= ncomp * M) return;
  const int64_t comp = q / M, i = q - comp * M;
  const double w = f ? f[(comp & 1) * fstride + i] : 1.0;
  const cplx v = cscale(t[q], w);
  acc[q] = first ? v : cadd(acc[q], v);
}
// W = A - v for the six planes
__global__ void k_cur_w(const double* A, const double* v, double* W, int64_t n) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q < n) W[q] = A[q] - v[q];
}
