// cluster3d.cuh -- H psi of a 32^3 spinor inside ONE thread-block cluster: the 3-D transforms never leave the chip.
//
// Eight CTAs (one per SM) form a cluster; CTA r keeps the x-planes 4r..4r+3 of two 32^3 complex buffers in its
// shared memory (8 padded 32 x 33 tiles, 132 KB), so the cluster holds 1 MB of lattice data:
//   Eq. 14: the buffers are the two components u, v of the spinor;
//   Eq. 40: the buffers are w and alpha_c * w of ONE component c, and the spinor takes two rounds.
// One round is
//   1. load the planes from global memory (coalesced, lane = z), FFT y and z in registers (regfft.cuh), leave the
//      plane spectrum [kz][ky] in the tile;
//   2. cluster barrier; every thread takes one x-line (kz, ky) of one buffer: its 32 points sit in the shared
//      memory of the 8 CTAs (distributed shared memory, 512-byte rows per warp), FFT x, times -k^2 / M
//      (Eq. 26), inverse FFT x, written back in place;
//   3. cluster barrier; inverse plane transforms, then the pointwise BdG mix (Eqs. 5, 15), the eps_n / norm
//      partial sums (Eq. 44b) and the stage combination of Alg. 2 exactly as pass C of fast3d.cuh.
// Global memory sees psi (and C_part) in and the result out; the spectra of fast3d.cuh / mega3d.cuh (12-14 MB of
// L2 traffic per spinor) do not exist.  Drop-in replacement of passes A, B, C of f3_hpsi (fast_step.cuh).
#pragma once
#include <cooperative_groups.h>
#include "fast3d.cuh"

namespace cg = cooperative_groups;

#define C3_CS 8                    // CTAs per cluster
#define C3_NT 256                  // threads per CTA: one warp per tile
#define C3_SMEM (8 * F3_TILE_BYTES)

struct C3Args {
  const cplx* psi;            // chunk base, [cnt][2][32][32][32]
  const double* scale;        // nullable
  const double* kperp2;       // per spinor of the chunk
  F3Fields F;
  const double *ky2, *kz2;    // natural order, Nyquist kept
  double kx2[32];
  double invM, kappa;
  cplx* out;                  // APPLY: H psi;  CORR: X = C_part - i kappa H psi;  RHS: Y = -i H psi
  const cplx* cpart;          // CORR
  double* part;               // [F3_NPART][cnt * 32]
  int cnt;
};

template <bool SYM, int MODE>
__global__ void __cluster_dims__(C3_CS, 1, 1) __launch_bounds__(C3_NT, 1) k_c3_hpsi(C3Args a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ double red[8 * F3_NPART];
  cplx* tiles = reinterpret_cast<cplx*>(smem_raw);
  cg::cluster_group cl = cg::this_cluster();
  constexpr int TILE = F3_N * F3_PITCH;
  const int r = (int)cl.block_rank();
  const int cid = blockIdx.x / C3_CS, ncl = gridDim.x / C3_CS;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int b = warp >> 2, xl = warp & 3;                     // phases 1-3: this warp's tile = (buffer b, local plane xl)
  const int ix = 4 * r + xl;                                  // its x-plane; in phase 2 the same number is its kz row
  const size_t M = (size_t)F3_N * F3_PLANE, pl = (size_t)ix * F3_PLANE;
  const int np = a.cnt * F3_N;
  cplx* T = tiles + warp * TILE;
  cplx* rem[C3_CS];                                           // this thread's x-line: 4 points in each CTA of the cluster
#pragma unroll
  for (int k = 0; k < C3_CS; ++k) rem[k] = cl.map_shared_rank(tiles + (b * 4) * TILE + ix * F3_PITCH + lane, k);
  const double kyz2 = a.ky2[lane] + a.kz2[ix];
  cplx x[F3_N];
#pragma unroll 1
  for (int n = cid; n < a.cnt; n += ncl) {
    const double s = a.scale ? a.scale[n] : 1.0, kp2 = a.kperp2[n];
    const cplx* pu = a.psi + (size_t)(2 * n) * M + pl;
    const cplx* pv = pu + M;
    double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
#pragma unroll 1
    for (int c = 0; c < (SYM ? 2 : 1); ++c) {
      F3_T0();
      // ---- 1. load + forward plane transform -------------------------------------------------------------
      {
        const int comp = SYM ? c : b;
        const cplx* src = comp ? pv : pu;
        const double* al = a.F.alpha[comp] + pl;
#pragma unroll
        for (int j = 0; j < F3_N; ++j) {
          double f = s;
          if (SYM && b) f *= al[j * F3_N + lane];
          x[j] = cscale(src[j * F3_N + lane], f);                // (y = j, z = lane)
        }
        F3_T(5, 0);
        f3_plane_forward(x, T, lane);                            // (kz = j, ky = lane)
#pragma unroll
        for (int j = 0; j < F3_N; ++j) T[j * F3_PITCH + lane] = x[j];
      }
      F3_T(5, 1);
      cl.sync();
      F3_T(5, 2);
      // ---- 2. x-lines through distributed shared memory ---------------------------------------------------
      {
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = rem[j >> 2][(j & 3) * TILE];
        F3_T(5, 3);
#pragma unroll 1
        for (int dir = 0; dir < 2; ++dir) {
          fft_reg<F3_N, false>(x);
#pragma unroll
          for (int j = 0; j < F3_N; ++j) {
            const double f = dir ? 1.0 : -(a.kx2[j] + kyz2) * a.invM;
            x[j] = make_double2(x[j].x * f, -x[j].y * f);
          }
        }
        F3_T(5, 4);
#pragma unroll
        for (int j = 0; j < F3_N; ++j) rem[j >> 2][(j & 3) * TILE] = x[j];
      }
      F3_T(5, 5);
      cl.sync();
      F3_T(5, 6);
      // ---- 3. inverse plane transform --------------------------------------------------------------------
      {
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = cconj(T[j * F3_PITCH + lane]);
        __syncwarp();
        f3_plane_forward(x, T, lane);                            // conj of the value at (y = j, z = lane)
        const double* al = a.F.alpha[c] + pl;
#pragma unroll
        for (int j = 0; j < F3_N; ++j) {
          const double f = (SYM && b == 0) ? al[j * F3_N + lane] : 1.0;
          T[j * F3_PITCH + lane] = make_double2(x[j].x * f, -x[j].y * f);
        }
      }
      F3_T(6, 0);
      __syncthreads();
      F3_T(6, 1);
      // ---- epilogue: warp = (plane xl, half b of its rows), both buffers of the plane ------------------------
      {
        const cplx* T0 = tiles + xl * TILE;
        const cplx* T1 = tiles + (4 + xl) * TILE;
        const cplx* dl = a.F.delta + pl;
        const cplx* dx = a.F.dext + pl;
#pragma unroll 1
        for (int jj0 = 0; jj0 < 16; jj0 += 4) {
          cplx gu[4], gv[4], gd[4], ge[4], g0[4], g1[4];
          double ga[4], gl[4], gU[4], gW[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int i = (16 * b + jj0 + q) * F3_N + lane;
            gu[q] = pu[i]; gv[q] = pv[i]; gd[q] = dl[i]; ge[q] = dx[i];
            if (SYM) { ga[q] = a.F.alpha[c][pl + i]; gl[q] = a.F.lap[c][pl + i]; gU[q] = a.F.U[c][pl + i]; }
            else { gU[q] = a.F.U[0][pl + i]; gW[q] = a.F.U[1][pl + i]; }
            if (MODE == F3_CORR) {
              if (SYM) g0[q] = a.cpart[(size_t)(2 * n + c) * M + pl + i];
              else { g0[q] = a.cpart[(size_t)(2 * n) * M + pl + i]; g1[q] = a.cpart[(size_t)(2 * n + 1) * M + pl + i]; }
            }
          }
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int j = 16 * b + jj0 + q, i = j * F3_N + lane, si = j * F3_PITCH + lane;
            const cplx u = cscale(gu[q], s), v = cscale(gv[q], s);
            const cplx D = cadd(gd[q], ge[q]);
#pragma unroll
            for (int cc = 0; cc < (SYM ? 1 : 2); ++cc) {
              const int comp = SYM ? c : cc;
              const cplx w = comp ? v : u;
              cplx K;
              if (SYM) {
                const cplx L = T1[si], t = T0[si];
                const double h = 0.5 * ga[q] * kp2;
                K.x = -0.25 * (L.x + t.x - gl[q] * w.x) + h * w.x;          // Eq. 40 + transverse shift
                K.y = -0.25 * (L.y + t.y - gl[q] * w.y) + h * w.y;
              } else {
                const cplx L = cc ? T1[si] : T0[si];
                K.x = -0.5 * L.x + 0.5 * kp2 * w.x;                          // Eq. 14
                K.y = -0.5 * L.y + 0.5 * kp2 * w.y;
              }
              const double pot = (SYM ? gU[q] : (cc ? gW[q] : gU[q])) - a.F.mu[comp];
              cplx H;
              if (comp == 0) H = cadd(K, cadd(cscale(u, pot), cmul(D, v)));  // Eqs. 5, 15
              else H = csub(cmul(cconj(D), u), cadd(K, cscale(v, pot)));
              e += w.x * H.x + w.y * H.y;
              cplx o;
              if (MODE == F3_APPLY) o = H;
              else if (MODE == F3_RHS) o = make_double2(H.y, -H.x);          // -i H
              else {
                const cplx cp = (SYM || cc == 0) ? g0[q] : g1[q];
                o = make_double2(cp.x + a.kappa * H.y, cp.y - a.kappa * H.x);   // C_part - i kappa H
                xx += cabs2(o); xpr += o.x * w.x + o.y * w.y; xpi += o.x * w.y - o.y * w.x; pp += cabs2(w);
              }
              a.out[(size_t)(2 * n + comp) * M + pl + i] = o;
            }
          }
        }
      }
      F3_T(6, 2);
      __syncthreads();                                           // the tiles are rewritten by the next round
      F3_T(6, 3);
    }
    e = warp_sum(e);
    if (MODE == F3_CORR) { xx = warp_sum(xx); xpr = warp_sum(xpr); xpi = warp_sum(xpi); pp = warp_sum(pp); }
    if (lane == 0) {
      red[warp * F3_NPART] = e;
      if (MODE == F3_CORR) { red[warp * F3_NPART + 1] = xx; red[warp * F3_NPART + 2] = xpr; red[warp * F3_NPART + 3] = xpi; red[warp * F3_NPART + 4] = pp; }
    }
    __syncthreads();
    if (warp < 4 && lane < (MODE == F3_CORR ? F3_NPART : 1))
      a.part[lane * np + n * F3_N + ix] = red[warp * F3_NPART + lane] + red[(warp + 4) * F3_NPART + lane];
  }
}
