// mega3m.cuh -- the 32^3 axis-by-axis stage kernel with the line derivatives in the MATRIX form of Eq. 28b
// on the FP64 tensor instructions (mma.sync.m8n8k4.f64 = DMMA).
//
// The second derivative along one axis is a real symmetric circulant D2[i][j] = c[(i - j) mod 32],
// c[m] = -(1/32) sum_q k_q^2 cos(2 pi q m / 32) (Eq. 26 with the Nyquist mode kept: even derivative).
// One radix-2 fold halves the work: with e[k] = w[k] + w[k+16], o[k] = w[k] - w[k+16] (k < 16),
//   out[i] + out[i+16] = sum_k (c[i-k] + c[i-k+16]) e[k],   out[i] - out[i+16] = sum_k (c[i-k] - c[i-k+16]) o[k],
// two 16 x 16 real symmetric matrices Ce, Co (the 1/2 of the unfolding folded in).  D2 is real, so the real and the
// imaginary parts of a field are independent real columns.  Measured on this B200: DMMA runs at 36.7 TFLOP/s on the
// same pipe as DFMA (33.9), so the pipe time equals that of the register FFT of mega3s.cuh (~ 280 k vs 295 k cycles
// per spinor-stage) -- what the matrix form buys is an eighth of the issue slots, no transposition (a tile is
// contracted along either index straight from shared memory), and tasks of ~ 170 registers instead of 255, so that
// three CTAs (12 warps) fit an SM instead of two (8 warps).
//
// P item (spinor, x-plane): the planes of u, v (swizzled 16-byte chunks) and of alpha_a, alpha_b are brought into shared
// memory by cp.async; a warp task is (component c, rows {8 rb .. +7} u {16 + 8 rb ..}, columns {8 cb ..} u {16 + 8 cb ..}):
// (d_y^2 + d_z^2) of w and of alpha w for both parts in DMMA accumulators, Q_c = alpha (..) w + (..)(alpha w) straight
// from the accumulator fragments to the Q ring.
// XE item (spinor, y-row): the (x, z) slabs of u, v, alpha_a, alpha_b in the same tile formats; d_x^2 of w and alpha w by
// DMMA, then the pointwise epilogue of mega3s.cuh (Eqs. 5, 15, 40; the stage combination of Alg. 2) on the fragments.
#pragma once
#include "mega3s.cuh"

#define F3M_APITCH 36                                   // doubles per row of an alpha tile (both fragment patterns conflict-free)
#define F3M_PSI_BYTES (F3_N * F3_N * 16)                // one plane of one component, unpadded, XOR-swizzled
#define F3M_AL_BYTES (F3_N * F3M_APITCH * 8)
#define F3M_BUF_BYTES (2 * F3M_PSI_BYTES + 2 * F3M_AL_BYTES)
#ifndef F3M_DEFAULT_ON
#define F3M_DEFAULT_ON 0                                  // wslda_tuning.dmma_stage >= this selects the kernel (1: opt-in, 0: default)
#endif
#ifndef F3M_PREFETCH
#define F3M_PREFETCH 1                                   // XE items: L2 prefetch of the Q / C_part rows behind the tile loads (+2-3 %)
#endif
#ifndef F3M_OCC
#define F3M_OCC 3
#endif

__device__ __forceinline__ void f3m_dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void f3m_cp16(void* smem, const void* g) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(g) : "memory");
}
__device__ __forceinline__ void f3m_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void f3m_cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// chunk (16 bytes) index of point (row, col) in a swizzled 32 x 32 complex tile: both the (8 rows x 4 cols) and the
// (4 rows x 8 cols) fragment footprints of a quarter warp hit eight distinct 16-byte bank groups
__device__ __forceinline__ int f3m_sw(int row, int col) { return row * F3_N + (col ^ (((row & 1) << 2) | (row & 2))); }

// the eight DMMA of one k-block: both fields (w, alpha w), both parts, even and odd fold; DATA_IS_B: the matrix is the
// A operand (contraction along the tile's row index), else the B operand (along its column index)
template <bool DATA_IS_B>
__device__ __forceinline__ void f3m_kblock(double (&acc)[2][2][2][2], cplx w1, cplx w2, double a1, double a2, double me, double mo) {
  const cplx v1 = cscale(w1, a1), v2 = cscale(w2, a2);
  const double d[8] = {w1.x + w2.x, w1.x - w2.x, w1.y + w2.y, w1.y - w2.y, v1.x + v2.x, v1.x - v2.x, v1.y + v2.y, v1.y - v2.y};
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    double& c0 = acc[i >> 2][(i >> 1) & 1][i & 1][0];
    double& c1 = acc[i >> 2][(i >> 1) & 1][i & 1][1];
    if (DATA_IS_B) f3m_dmma(c0, c1, (i & 1) ? mo : me, d[i]); else f3m_dmma(c0, c1, d[i], (i & 1) ? mo : me);
  }
}

// loads of one (spinor, x-plane) [ROW = false: tile row = y] or of one (spinor, y-row) slab [ROW = true: tile row = x]:
// u, v tiles and the two alpha tiles, 128 threads, 16-byte cp.async
template <bool ROW>
__device__ __forceinline__ void f3m_load(const F3Mega& a, int n, int idx, unsigned char* buf) {
  const size_t M = (size_t)F3_N * F3_PLANE;
  const size_t o0 = ROW ? (size_t)idx * F3_N : (size_t)idx * F3_PLANE, rs = ROW ? F3_PLANE : F3_N;   // tile origin, row stride
#pragma unroll
  for (int c = 0; c < 2; ++c) {
    const cplx* src = a.psi + (size_t)(2 * n + c) * M + o0;
    cplx* T = reinterpret_cast<cplx*>(buf + c * F3M_PSI_BYTES);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const int i = k * 128 + threadIdx.x, row = i >> 5, col = i & 31;
      f3m_cp16(T + f3m_sw(row, col), src + (size_t)row * rs + col);
    }
    const double* al = a.F.alpha[c] + o0;
    double* AL = reinterpret_cast<double*>(buf + 2 * F3M_PSI_BYTES + c * F3M_AL_BYTES);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int i = k * 128 + threadIdx.x, row = i >> 4, c2 = (i & 15) * 2;
      f3m_cp16(AL + row * F3M_APITCH + c2, al + (size_t)row * rs + c2);
    }
  }
}

// one warp task of a P item; T, AL: this component's tiles; q: this component's plane of the Q ring
// CUR: the in-plane part of the current / velocity coupling (Eq. 4c, R27) rides on the alpha-w field's results: with the first-
// derivative matrices stored as 2 D (mat1), -1/4 [.. + (+-i)(W_d (2 D_d w) + 2 D_d (W_d w))] = .. + (+-)(-(i/2)){W_d, d_d} w; sgn = +1 for u, -1 for v
template <bool CUR = false>
__device__ __forceinline__ void f3m_task_p(const cplx* T, const double* AL, const double* mat, int rb, int cb, double s, cplx* q, uint64_t pol,
                                           const double* mat1 = nullptr, const double* Wy = nullptr, const double* Wz = nullptr, double sgn = 1.0) {
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  double mA[2][4], mB[2][4];                            // fragments of Ce, Co: rows of the y matrices (A operand), of the z matrices (B operand)
#pragma unroll
  for (int eo = 0; eo < 2; ++eo)
#pragma unroll
    for (int kb = 0; kb < 4; ++kb) {
      mA[eo][kb] = mat[(1 * 2 + eo) * 256 + (rb * 4 + kb) * 32 + lane];         // fragment order (ctx.cuh): [axis][Ce | Co][block][k-block][lane]
      mB[eo][kb] = mat[(0 * 2 + eo) * 256 + (cb * 4 + kb) * 32 + lane];
    }
  double out[2][2][2][2][2];                            // [field w | alpha w][re | im][row half][col half][j]
  // d_y^2: A = Ce / Co rows, B = folded data W[k = y][n = z]
#pragma unroll
  for (int zi = 0; zi < 2; ++zi) {
    const int z = 8 * cb + 16 * zi + g;
    double acc[2][2][2][2];                             // [field][part][E | O][j]
#pragma unroll
    for (int i = 0; i < 16; ++i) (&acc[0][0][0][0])[i] = 0.0;
#pragma unroll
    for (int kb = 0; kb < 4; ++kb) {
      const int y1 = 4 * kb + t, y2 = y1 + 16;
      f3m_kblock<true>(acc, T[f3m_sw(y1, z)], T[f3m_sw(y2, z)], AL[y1 * F3M_APITCH + z], AL[y2 * F3M_APITCH + z], mA[0][kb], mA[1][kb]);
    }
#pragma unroll
    for (int f = 0; f < 2; ++f)
#pragma unroll
      for (int p = 0; p < 2; ++p)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          out[f][p][0][zi][j] = acc[f][p][0][j] + acc[f][p][1][j];
          out[f][p][1][zi][j] = acc[f][p][0][j] - acc[f][p][1][j];
        }
    if (CUR) {                                              // W_y (2 D_y w) + 2 D_y (W_y w)
#pragma unroll
      for (int i = 0; i < 16; ++i) (&acc[0][0][0][0])[i] = 0.0;
#pragma unroll
      for (int kb = 0; kb < 4; ++kb) {
        const int y1 = 4 * kb + t, y2 = y1 + 16;
        f3m_kblock<true>(acc, T[f3m_sw(y1, z)], T[f3m_sw(y2, z)], __ldg(Wy + y1 * F3_N + z), __ldg(Wy + y2 * F3_N + z),
                         __ldg(mat1 + (1 * 2 + 0) * 256 + (rb * 4 + kb) * 32 + lane), __ldg(mat1 + (1 * 2 + 1) * 256 + (rb * 4 + kb) * 32 + lane));
      }
#pragma unroll
      for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const double sg = h ? -1.0 : 1.0, wv = __ldg(Wy + (8 * rb + 16 * h + g) * F3_N + 8 * cb + 16 * zi + 2 * t + j);
          const double tr = wv * (acc[0][0][0][j] + sg * acc[0][0][1][j]) + (acc[1][0][0][j] + sg * acc[1][0][1][j]);
          const double ti = wv * (acc[0][1][0][j] + sg * acc[0][1][1][j]) + (acc[1][1][0][j] + sg * acc[1][1][1][j]);
          out[1][0][h][zi][j] -= sgn * ti; out[1][1][h][zi][j] += sgn * tr;
        }
    }
  }
  // d_z^2: A = folded data W[m = y][k = z], B = Ce / Co columns
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int y = 8 * rb + 16 * h + g;
    double acc[2][2][2][2];
#pragma unroll
    for (int i = 0; i < 16; ++i) (&acc[0][0][0][0])[i] = 0.0;
#pragma unroll
    for (int kb = 0; kb < 4; ++kb) {
      const int z1 = 4 * kb + t, z2 = z1 + 16;
      f3m_kblock<false>(acc, T[f3m_sw(y, z1)], T[f3m_sw(y, z2)], AL[y * F3M_APITCH + z1], AL[y * F3M_APITCH + z2], mB[0][kb], mB[1][kb]);
    }
#pragma unroll
    for (int f = 0; f < 2; ++f)
#pragma unroll
      for (int p = 0; p < 2; ++p)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          out[f][p][h][0][j] += acc[f][p][0][j] + acc[f][p][1][j];
          out[f][p][h][1][j] += acc[f][p][0][j] - acc[f][p][1][j];
        }
    if (CUR) {                                              // W_z (2 D_z w) + 2 D_z (W_z w)
#pragma unroll
      for (int i = 0; i < 16; ++i) (&acc[0][0][0][0])[i] = 0.0;
#pragma unroll
      for (int kb = 0; kb < 4; ++kb) {
        const int z1 = 4 * kb + t, z2 = z1 + 16;
        f3m_kblock<false>(acc, T[f3m_sw(y, z1)], T[f3m_sw(y, z2)], __ldg(Wz + y * F3_N + z1), __ldg(Wz + y * F3_N + z2),
                          __ldg(mat1 + (0 * 2 + 0) * 256 + (cb * 4 + kb) * 32 + lane), __ldg(mat1 + (0 * 2 + 1) * 256 + (cb * 4 + kb) * 32 + lane));
      }
#pragma unroll
      for (int zi = 0; zi < 2; ++zi)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const double sg = zi ? -1.0 : 1.0, wv = __ldg(Wz + y * F3_N + 8 * cb + 16 * zi + 2 * t + j);
          const double tr = wv * (acc[0][0][0][j] + sg * acc[0][0][1][j]) + (acc[1][0][0][j] + sg * acc[1][0][1][j]);
          const double ti = wv * (acc[0][1][0][j] + sg * acc[0][1][1][j]) + (acc[1][1][0][j] + sg * acc[1][1][1][j]);
          out[1][0][h][zi][j] -= sgn * ti; out[1][1][h][zi][j] += sgn * tr;
        }
    }
  }
  // Q_c = s [ alpha (d_y^2 + d_z^2) w + (d_y^2 + d_z^2)(alpha w) ] at (y = 8 rb + 16 h + g, z = 8 cb + 16 zi + 2 t + j)
#pragma unroll
  for (int h = 0; h < 2; ++h)
#pragma unroll
    for (int zi = 0; zi < 2; ++zi) {
      const int y = 8 * rb + 16 * h + g, z = 8 * cb + 16 * zi + 2 * t;
      const double2 al = *reinterpret_cast<const double2*>(AL + y * F3M_APITCH + z);
      st_pol(q + y * F3_N + z, make_double2(s * (al.x * out[0][0][h][zi][0] + out[1][0][h][zi][0]), s * (al.x * out[0][1][h][zi][0] + out[1][1][h][zi][0])), pol);
      st_pol(q + y * F3_N + z + 1, make_double2(s * (al.y * out[0][0][h][zi][1] + out[1][0][h][zi][1]), s * (al.y * out[0][1][h][zi][1] + out[1][1][h][zi][1])), pol);
    }
}

struct F3MMega {
  F3Mega m;                      // spec0 = Q ring [R][gs][2][M]
  int pm, em;                    // x-planes per P item, y-rows per XE item
  const double* mat;             // [axis z, y, x][Ce | Co][16][16]
  const double* mat1;            // CUR: the first-derivative matrices (2 D, folded), same layout
  const double* curW;            // CUR: W_sigma,d = A_sigma,d - v_ext,sigma,d, [2][3][M]
};

// ---- P item: pm x-planes of one spinor -----------------------------------------------------------------------------
template <bool CUR = false>
__device__ __forceinline__ void f3m_body_p(const F3MMega& A, const F3Pol& pol, int g, int ip, unsigned char* buf) {
  const F3Mega& a = A.m;
  const int warp = threadIdx.x >> 5;
  const int per = F3_N / A.pm, nl = ip / per, ix0 = (ip - nl * per) * A.pm, n = g * a.gs + nl;
  if (n >= a.n) return;
  const size_t M = (size_t)F3_N * F3_PLANE;
  const double s = a.scale ? a.scale[n] : 1.0;
  const int c = warp >> 1, rb = warp & 1;
  const cplx* T = reinterpret_cast<const cplx*>(buf + c * F3M_PSI_BYTES);
  const double* AL = reinterpret_cast<const double*>(buf + 2 * F3M_PSI_BYTES + c * F3M_AL_BYTES);
  for (int k = 0; k < A.pm; ++k) {
    const int ix = ix0 + k;
    f3m_load<false>(a, n, ix, buf);
    f3m_cp_commit();
    f3m_cp_wait<0>();
    __syncthreads();
    cplx* q = a.spec0 + (((size_t)(g % F3_RING) * a.gs + nl) * 2 + c) * M + (size_t)ix * F3_PLANE;
#pragma unroll 1
    for (int cb = 0; cb < 2; ++cb) {
      if (CUR) {
        const double* W = A.curW + (size_t)(c * 3) * M + (size_t)ix * F3_PLANE;       // W_c,x | + M: W_c,y | + 2 M: W_c,z of this plane
        f3m_task_p<true>(T, AL, A.mat, rb, cb, s, q, pol.keep, A.mat1, W + M, W + 2 * M, c ? -1.0 : 1.0);
      } else f3m_task_p(T, AL, A.mat, rb, cb, s, q, pol.keep);
    }
    __syncthreads();
  }
}

// ---- XE item: em y-rows of one spinor.  A warp task is (rows {8 rb ..} u {16 + 8 rb ..} of x, 8 columns of z) for BOTH
// components: d_x^2 of w and alpha w by DMMA, then the pointwise epilogue on the accumulator fragments ------------------
template <int MODE, bool CUR = false>
__device__ __forceinline__ void f3m_body_xe(const F3MMega& A, const F3Pol& pol, int g, int ie, unsigned char* buf, double* red) {
  const F3Mega& a = A.m;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, gq = lane >> 2, t = lane & 3;
  const int per = F3_N / A.em, nl = ie / per, y0 = (ie - nl * per) * A.em, n = g * a.gs + nl;
  if (n >= a.n) return;
  const size_t M = (size_t)F3_N * F3_PLANE;
  const size_t ring = ((size_t)(g % F3_RING) * a.gs + nl) * 2;
  const double s = a.scale ? a.scale[n] : 1.0, kp2 = a.kperp2[n];
  const int rb = warp & 1;
  double mA[2][4];
#pragma unroll
  for (int eo = 0; eo < 2; ++eo)
#pragma unroll
    for (int kb = 0; kb < 4; ++kb) mA[eo][kb] = A.mat[(2 * 2 + eo) * 256 + (rb * 4 + kb) * 32 + lane];
  const cplx* Tu = reinterpret_cast<const cplx*>(buf);
  const cplx* Tv = reinterpret_cast<const cplx*>(buf + F3M_PSI_BYTES);
  const double* ALa = reinterpret_cast<const double*>(buf + 2 * F3M_PSI_BYTES);
  const double* ALb = reinterpret_cast<const double*>(buf + 2 * F3M_PSI_BYTES + F3M_AL_BYTES);
  cplx* ou = (MODE == F3_APPLY ? a.out + (size_t)(2 * n) * M : a.X + ring * M);
  for (int k = 0; k < A.em; ++k) {
    const int y = y0 + k;
    f3m_load<true>(a, n, y, buf);
    f3m_cp_commit();
    double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
#if F3M_PREFETCH
    // the rows of Q (and C_part) this CTA's epilogue reads: 32 x-rows of 512 bytes per component; one 128-byte line per thread
    {
      const int xr = threadIdx.x >> 2, seg = threadIdx.x & 3;
      const size_t i = (size_t)y * F3_N + (size_t)xr * F3_PLANE + seg * 8;
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        f3_pf(a.spec0 + (ring + c) * M + i);
        if (MODE == F3_CORR) f3_pf(a.cpart + (size_t)(2 * n + c) * M + i);
      }
    }
#endif
    f3m_cp_wait<0>();
    __syncthreads();
#pragma unroll 1
    for (int ci = 0; ci < 2; ++ci) {
      const int cb = (warp >> 1) + 2 * ci, z = 8 * cb + gq;
      const size_t off = (size_t)y * F3_N + 8 * cb + 2 * t;      // + x * F3_PLANE + j
      // epilogue inputs that do not depend on the transforms: issued first
      cplx Qr[2][2][2], Cr[2][2][2], pq[2][2], pD[2][2];        // [component][row half][j], [row half][j]
#pragma unroll
      for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const size_t i = off + (size_t)(8 * rb + 16 * h + gq) * F3_PLANE + j;
          pq[h][j] = a.pack[i]; pD[h][j] = a.pack[M + i];
#pragma unroll
          for (int c = 0; c < 2; ++c) {
            Qr[c][h][j] = ld_pol(a.spec0 + (ring + c) * M + i, pol.drop);
            if (MODE == F3_CORR) Cr[c][h][j] = ld_pol(a.cpart + (size_t)(2 * n + c) * M + i, pol.drop);
          }
        }
      cplx L[2][2][2];                                          // s [alpha d_x^2 w + d_x^2 (alpha w)]: [component][row half][j]
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const cplx* T = c ? Tv : Tu;
        const double* AL = c ? ALb : ALa;
        double acc[2][2][2][2];                                 // [field][part][E | O][j]
#pragma unroll
        for (int i = 0; i < 16; ++i) (&acc[0][0][0][0])[i] = 0.0;
#pragma unroll
        for (int kb = 0; kb < 4; ++kb) {
          const int x1 = 4 * kb + t, x2 = x1 + 16;
          f3m_kblock<true>(acc, T[f3m_sw(x1, z)], T[f3m_sw(x2, z)], AL[x1 * F3M_APITCH + z], AL[x2 * F3M_APITCH + z], mA[0][kb], mA[1][kb]);
        }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const double2 al = *reinterpret_cast<const double2*>(AL + (8 * rb + 16 * h + gq) * F3M_APITCH + 8 * cb + 2 * t);
          const double sg = h ? -1.0 : 1.0;
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            const double aj = j ? al.y : al.x;
            const double wr = acc[0][0][0][j] + sg * acc[0][0][1][j], wi = acc[0][1][0][j] + sg * acc[0][1][1][j];
            const double vr = acc[1][0][0][j] + sg * acc[1][0][1][j], vi = acc[1][1][0][j] + sg * acc[1][1][1][j];
            L[c][h][j] = make_double2(s * (aj * wr + vr), s * (aj * wi + vi));
          }
        }
        if (CUR) {                                              // the x part of the coupling: W_x (2 D_x w) + 2 D_x (W_x w), rotated by +-i
          const double* Wx = A.curW + (size_t)(c * 3) * M + (size_t)y * F3_N;          // + x * F3_PLANE + z
#pragma unroll
          for (int i = 0; i < 16; ++i) (&acc[0][0][0][0])[i] = 0.0;
#pragma unroll
          for (int kb = 0; kb < 4; ++kb) {
            const int x1 = 4 * kb + t, x2 = x1 + 16;
            f3m_kblock<true>(acc, T[f3m_sw(x1, z)], T[f3m_sw(x2, z)], __ldg(Wx + (size_t)x1 * F3_PLANE + z), __ldg(Wx + (size_t)x2 * F3_PLANE + z),
                             __ldg(A.mat1 + (2 * 2 + 0) * 256 + (rb * 4 + kb) * 32 + lane), __ldg(A.mat1 + (2 * 2 + 1) * 256 + (rb * 4 + kb) * 32 + lane));
          }
          const double sgn = c ? -1.0 : 1.0;
#pragma unroll
          for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              const double sg = h ? -1.0 : 1.0, wv = __ldg(Wx + (size_t)(8 * rb + 16 * h + gq) * F3_PLANE + 8 * cb + 2 * t + j);
              const double tr = wv * (acc[0][0][0][j] + sg * acc[0][0][1][j]) + (acc[1][0][0][j] + sg * acc[1][0][1][j]);
              const double ti = wv * (acc[0][1][0][j] + sg * acc[0][1][1][j]) + (acc[1][1][0][j] + sg * acc[1][1][1][j]);
              L[c][h][j].x -= s * sgn * ti; L[c][h][j].y += s * sgn * tr;
            }
        }
      }
      // pointwise epilogue at (x = 8 rb + 16 h + gq, z = 8 cb + 2 t + j): Eqs. 5, 15, 40; the stage combination
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int x = 8 * rb + 16 * h + gq;
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const int zz = 8 * cb + 2 * t + j;
          const size_t i = off + (size_t)x * F3_PLANE + j;
          const cplx qq = pq[h][j], D = pD[h][j];
          const cplx u = cscale(Tu[f3m_sw(x, zz)], s), v = cscale(Tv[f3m_sw(x, zz)], s);
          const double ha = 0.5 * kp2 * ALa[x * F3M_APITCH + zz], hb = 0.5 * kp2 * ALb[x * F3M_APITCH + zz];
          const cplx Lu = cadd(L[0][h][j], Qr[0][h][j]), Lv = cadd(L[1][h][j], Qr[1][h][j]);
          const cplx Ku = make_double2(-0.25 * Lu.x + ha * u.x, -0.25 * Lu.y + ha * u.y);
          const cplx Kv = make_double2(-0.25 * Lv.x + hb * v.x, -0.25 * Lv.y + hb * v.y);
          const cplx Hu = cadd(Ku, cadd(cscale(u, qq.x), cmul(D, v)));
          const cplx Hv = csub(cmul(cconj(D), u), cadd(Kv, cscale(v, qq.y)));
          e += u.x * Hu.x + u.y * Hu.y + v.x * Hv.x + v.y * Hv.y;
          if (MODE == F3_APPLY) { st_pol_nb(ou + i, Hu, pol.drop); st_pol_nb(ou + M + i, Hv, pol.drop); }
          else if (MODE == F3_RHS) {
            st_pol_nb(ou + i, make_double2(Hu.y, -Hu.x), pol.keep); st_pol_nb(ou + M + i, make_double2(Hv.y, -Hv.x), pol.keep);
          } else {
            const cplx xu = make_double2(Cr[0][h][j].x + a.kappa * Hu.y, Cr[0][h][j].y - a.kappa * Hu.x);
            const cplx xv = make_double2(Cr[1][h][j].x + a.kappa * Hv.y, Cr[1][h][j].y - a.kappa * Hv.x);
            st_pol_nb(ou + i, xu, pol.keep); st_pol_nb(ou + M + i, xv, pol.keep);
            xx += cabs2(xu) + cabs2(xv);
            xpr += xu.x * u.x + xu.y * u.y + xv.x * v.x + xv.y * v.y;
            xpi += xu.x * u.y - xu.y * u.x + xv.x * v.y - xv.y * v.x;
            pp += cabs2(u) + cabs2(v);
          }
        }
      }
    }
    e = warp_sum(e);
    if (MODE == F3_CORR) { xx = warp_sum(xx); xpr = warp_sum(xpr); xpi = warp_sum(xpi); pp = warp_sum(pp); }
    if (lane == 0) {
      double* q = red + warp * F3_NPART;
      q[0] = e;
      if (MODE == F3_CORR) { q[1] = xx; q[2] = xpr; q[3] = xpi; q[4] = pp; }
    }
    __syncthreads();                                            // the tiles are free again; the partial sums are in place
    if (threadIdx.x < (MODE == F3_CORR ? F3_NPART : 1)) {
      const size_t np = (size_t)a.n * F3_N, o = (size_t)n * F3_N + y;
      const int p = threadIdx.x;
      a.part[p * np + o] = (red[p] + red[F3_NPART + p]) + (red[2 * F3_NPART + p] + red[3 * F3_NPART + p]);
    }
    __syncthreads();
  }
}

// tick t: P(t), XE(t-1), D(t-2): the dispatch of k_f3s_mega (mega3s.cuh) with the matrix-form bodies
template <int MODE, bool CUR = false>
__global__ void __launch_bounds__(128, CUR ? 2 : F3M_OCC) k_f3m_mega(F3MMega A) {
  extern __shared__ __align__(128) unsigned char f3m_buf[];
  __shared__ int s_item[2];
  __shared__ double s_eps[32], s_sn[32], red[4 * F3_NPART];
  const F3Mega& a = A.m;
  const F3Pol pol = f3_policies();
  const int G = a.G;
  int* done = reinterpret_cast<int*>(a.sync + 1);
  const int nP = a.gs * F3_N / A.pm, nE = a.gs * F3_N / A.em, nD = MODE == F3_APPLY ? 0 : F3_N * F3_DSPLIT;
  const int IT = nP + nE + nD, total = (G + 2) * IT;
  int t1 = 0;
  if (threadIdx.x == 0) t1 = atomicAdd(&a.sync->next, 1);
  for (;;) {
    if (threadIdx.x == 0) s_item[0] = t1;
    __syncthreads();
    const int item = s_item[0];
    __syncthreads();
    if (item >= total) break;
    const int tick = item / IT, r = item - tick * IT;
    bool drew = false;
    if (r < nP) {
      const int g = tick;
      if (g < G) {
        if (g >= F3_RING) f3_wait(&done[G + g - F3_RING], nE, a.sync);                 // the Q slot is free
        f3m_body_p<CUR>(A, pol, g, r, f3m_buf);
        f3_signal(&done[g], &a.sync->next, t1); drew = true;
      }
    } else if (r < nP + nE) {
      const int g = tick - 1;
      if (g >= 0 && g < G) {
        f3_wait(&done[g], nP, a.sync);
        if (MODE != F3_APPLY && g >= F3_RING) f3_wait(&done[2 * G + g - F3_RING], nD, a.sync);   // the X slot is free
        f3m_body_xe<MODE, CUR>(A, pol, g, r - nP, f3m_buf, red);
        f3_signal(&done[G + g], &a.sync->next, t1); drew = true;
      }
    } else {
      const int g = tick - 2;
      if (g >= 0 && g < G) {
        f3_wait(&done[G + g], nE, a.sync);
        if (g >= F3_RING) f3_wait(&done[2 * G + g - F3_RING], nD, a.sync);             // the density slot
        if (MODE != F3_APPLY) f3_body_d<MODE>(a, pol, g, r - nP - nE, s_eps, s_sn);
        f3_signal(&done[2 * G + g], &a.sync->next, t1); drew = true;
      }
    }
    if (!drew && threadIdx.x == 0) t1 = atomicAdd(&a.sync->next, 1);
  }
}
