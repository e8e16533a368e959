// onchip_step.cuh -- fused ABM stage kernels for lattices whose spinors fit in shared memory (M <= 4096 points:
// the quasi-1D / quasi-2D modes and small 3-D boxes; configs[0..2]) with the Eq. 14 kinetic operator.
// A CTA keeps a batch of S spinors (S * 2 * M <= 8192 complex128 = 128 KB) on chip for the whole stage:
//   load psi -> forward FFT over the held axes -> -k^2/M (Eq. 26) -> inverse FFT, all in place,
//   pointwise BdG mix (Eqs. 5, 15) -> eps_n = Re <psi|H psi> reduced inside the CTA (Eq. 44b) ->
//   RHS : f = -i (H - eps) psi written once                                        (Alg. 2 step 9)
//   CORR: phi_new = C_part + c0 dt f, its norm reduced inside the CTA, normalised, written once over P,
//         and the densities of phi_new accumulated per CTA in registers             (Alg. 2 steps 3-4, 8)
// so a stage is ONE HBM round trip (read psi [+ C_part], write the result) with no scratch traffic at all.
// Density partials [CTA][4][slots] are summed in a fixed order afterwards: bit-reproducible.
#pragma once
#include "ops.cuh"

enum { OC_APPLY = 0, OC_CORR = 1, OC_RHS = 2 };
#define OC_MAXS 64              // spinors per CTA batch (s_eps / s_sn arrays)
#define OC_SLOTS 8              // (lattice point, spinor) pairs per thread and batch

struct OCArgs {
  Lat L;
  const cplx* psi;             // [n][2][M], first spinor of the call
  const double* scale;         // per spinor, nullable
  const double* kperp2;
  Fields F;
  cplx* out;                   // APPLY: H psi; RHS: f; CORR: phi_new (may alias psi)
  const cplx* cpart;
  double kappa, dV;
  int use_shift, normalize;
  double* eps_out;             // nullable: true eps_n
  int do_dens;
  const double *cpref, *w_a, *w_b;
  double* dpart;               // [gridDim.x][4][slots], slots = max(M, 256)
  int64_t n;
  int S;
  int dm;                      // 64 x 64: Laplacian in matrix form on DMMA (storage index swizzled: oc_ix)
  const double* curW;          // current / velocity coupling (DM = 1 only): W_sigma,d = A_sigma,d - v_ext,sigma,d, [2][3][M]; nullable
  const double* mat;           // [axis][Ce | Co][32][32]
};

// per-spinor sums of E[s][i] over the lattice: warp w takes spinors w, w + 8, ...; fixed order
__device__ __forceinline__ void oc_reduce(const double* E, int cnt, int lgM, double* out_s) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, M = 1 << lgM;
  for (int s = warp; s < cnt; s += (blockDim.x >> 5)) {
    double v = 0.0;
    for (int i = lane; i < M; i += 32) v += E[(s << lgM) + i];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) out_s[s] = v;
  }
}
// one spinor of 4096 points, 16 warps: every warp sums a slice of 256, warp 0 adds the 16 slices in index order.
// Contains the barrier between the two levels; `scratch` = 16 doubles of shared memory.
__device__ __forceinline__ void oc_reduce1(const double* E, double* scratch, double* out_s) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double v = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) v += E[warp * 256 + k * 32 + lane];
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if (lane == 0) scratch[warp] = v;
  __syncthreads();
  if (warp == 0) {
    double t = lane < 16 ? scratch[lane] : 0.0;
    for (int o = 8; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) out_s[0] = t;
  }
}

template <int MAXPT>
__device__ __forceinline__ void oc_dens_acc(double (&acc)[MAXPT][4], int w, int PT, double a0, double a1, double a2, double a3) {
#pragma unroll
  for (int kk = 0; kk < MAXPT; ++kk)
    if ((w & (PT - 1)) == kk) { acc[kk][0] += a0; acc[kk][1] += a1; acc[kk][2] += a2; acc[kk][3] += a3; }
}

// MAXPT = compile-time bound on the lattice points per thread, max(1, M / blockDim.x): 2 (256 threads, M <= 512,
// two CTAs per SM) or 8 (512 threads for M up to 4096, one CTA per SM)
// ---- 64 x 64 (quasi-2D, configs[2]): the Laplacian in the matrix form of Eq. 28b on FP64 tensor
// instructions.  d^2 along an axis is a real symmetric circulant; folded once (e = w[k] + w[k+32], o = w[k] - w[k+32]) it is
// two 32 x 32 real matrices Ce, Co with out[i] +- out[i+32] = Ce e +- Co o.  A warp owns rows {8 rb ..} u {32 + 8 rb ..} by
// columns {8 cb ..} u {32 + 8 cb ..} (16 warps = 16 blocks), contracts the tile along its rows (matrix = A operand) and along
// its columns (matrix = B operand) straight from shared memory, and keeps its 16 x 16 results in accumulator fragments until
// every warp has read the tile; then the tile is overwritten in place.  No transform passes, no spectrum, two barriers.
// The tile's 16-byte elements are stored at oc_ix(i): column ^ f(row), conflict-free for both fragment footprints.
// (DM = 1: 64 x 64 tile, column ^ f(row); DM = 2: lines of 128 points, point ^ 4 on odd lines; DM = 0: natural order)
__device__ __forceinline__ int oc_ix(int line, int i, int dm) {
  return dm == 1 ? i ^ ((((i >> 6) & 1) << 2) | ((i >> 6) & 2)) : dm == 2 ? i ^ ((line & 1) << 2) : i;
}
__device__ __forceinline__ void oc_dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void oc_lap64(const cplx* T, const double* mat, int rb, int cb, double (&out)[2][2][2][2]) {   // [re | im][h][zi][j]
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  // matrices in fragment order (ctx.cuh): [axis][Ce | Co][block][k-block][lane]
  const double* mx = mat + rb * 256 + lane;                     // rows of Cx (A operand): + eo * 1024 + 32 kb
  const double* my = mat + 2048 + cb * 256 + lane;              // columns of Cy = its rows (symmetric) (B operand)
#pragma unroll
  for (int zi = 0; zi < 2; ++zi) {                              // contraction along the rows: (d_x^2 w)[i][z]
    const int z = 8 * cb + 32 * zi + g;
    double acc[2][2][2] = {};                                   // [re | im][E | O][j]
#pragma unroll
    for (int kb = 0; kb < 8; ++kb) {
      const int x1 = 4 * kb + t;
      const cplx w1 = T[oc_ix(0, x1 * 64 + z, 1)], w2 = T[oc_ix(0, (x1 + 32) * 64 + z, 1)];
      const double me = __ldg(mx + 32 * kb), mo = __ldg(mx + 1024 + 32 * kb);
      oc_dmma(acc[0][0][0], acc[0][0][1], me, w1.x + w2.x); oc_dmma(acc[0][1][0], acc[0][1][1], mo, w1.x - w2.x);
      oc_dmma(acc[1][0][0], acc[1][0][1], me, w1.y + w2.y); oc_dmma(acc[1][1][0], acc[1][1][1], mo, w1.y - w2.y);
    }
#pragma unroll
    for (int p = 0; p < 2; ++p)
#pragma unroll
      for (int j = 0; j < 2; ++j) { out[p][0][zi][j] = acc[p][0][j] + acc[p][1][j]; out[p][1][zi][j] = acc[p][0][j] - acc[p][1][j]; }
  }
#pragma unroll
  for (int h = 0; h < 2; ++h) {                                 // contraction along the columns: (d_y^2 w)[x][i]
    const int x = 8 * rb + 32 * h + g;
    double acc[2][2][2] = {};
#pragma unroll
    for (int kb = 0; kb < 8; ++kb) {
      const int y1 = 4 * kb + t;
      const cplx w1 = T[oc_ix(0, x * 64 + y1, 1)], w2 = T[oc_ix(0, x * 64 + y1 + 32, 1)];
      const double me = __ldg(my + 32 * kb), mo = __ldg(my + 1024 + 32 * kb);
      oc_dmma(acc[0][0][0], acc[0][0][1], w1.x + w2.x, me); oc_dmma(acc[0][1][0], acc[0][1][1], w1.x - w2.x, mo);
      oc_dmma(acc[1][0][0], acc[1][0][1], w1.y + w2.y, me); oc_dmma(acc[1][1][0], acc[1][1][1], w1.y - w2.y, mo);
    }
#pragma unroll
    for (int p = 0; p < 2; ++p)
#pragma unroll
      for (int j = 0; j < 2; ++j) { out[p][h][0][j] += acc[p][0][j] + acc[p][1][j]; out[p][h][1][j] += acc[p][0][j] - acc[p][1][j]; }
  }
}
// The current / velocity coupling of Eq. 4c in the Hermitian form of DESIGN R27 on the same tile: adds
//   rot * [ W_x (D_x w) + D_x (W_x w) + W_y (D_y w) + D_y (W_y w) ]
// to `out`, D_d the spectral FIRST derivative as a folded circulant (odd derivative: Nyquist mode dropped),
// W_d real fields [64][64] in global memory (L1 / L2).  rot = +i (sgn = +1: component u, so that -1/2 out carries
// -(i/2){W, grad} u) or -i (sgn = -1: component v, whose coupling enters -h_b^* with the opposite sign).
__device__ __forceinline__ void oc_cur64(const cplx* T, const double* mat1, const double* Wx, const double* Wy, int rb, int cb, double sgn,
                                         double (&out)[2][2][2][2]) {
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const double* mx = mat1 + rb * 256 + lane;
  const double* my = mat1 + 2048 + cb * 256 + lane;
#pragma unroll
  for (int zi = 0; zi < 2; ++zi) {                              // along the rows: D_x
    const int z = 8 * cb + 32 * zi + g;
    double aG[2][2][2] = {}, aH[2][2][2] = {};                  // [re | im][E | O][j]: D_x w and D_x (W_x w)
#pragma unroll
    for (int kb = 0; kb < 8; ++kb) {
      const int x1 = 4 * kb + t;
      const cplx w1 = T[oc_ix(0, x1 * 64 + z, 1)], w2 = T[oc_ix(0, (x1 + 32) * 64 + z, 1)];
      const cplx h1 = cscale(w1, __ldg(Wx + x1 * 64 + z)), h2 = cscale(w2, __ldg(Wx + (x1 + 32) * 64 + z));
      const double me = __ldg(mx + 32 * kb), mo = __ldg(mx + 1024 + 32 * kb);
      oc_dmma(aG[0][0][0], aG[0][0][1], me, w1.x + w2.x); oc_dmma(aG[0][1][0], aG[0][1][1], mo, w1.x - w2.x);
      oc_dmma(aG[1][0][0], aG[1][0][1], me, w1.y + w2.y); oc_dmma(aG[1][1][0], aG[1][1][1], mo, w1.y - w2.y);
      oc_dmma(aH[0][0][0], aH[0][0][1], me, h1.x + h2.x); oc_dmma(aH[0][1][0], aH[0][1][1], mo, h1.x - h2.x);
      oc_dmma(aH[1][0][0], aH[1][0][1], me, h1.y + h2.y); oc_dmma(aH[1][1][0], aH[1][1][1], mo, h1.y - h2.y);
    }
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const double sg = h ? -1.0 : 1.0;
        const double wv = __ldg(Wx + (8 * rb + 32 * h + g) * 64 + 8 * cb + 32 * zi + 2 * t + j);
        const double tr = wv * (aG[0][0][j] + sg * aG[0][1][j]) + (aH[0][0][j] + sg * aH[0][1][j]);
        const double ti = wv * (aG[1][0][j] + sg * aG[1][1][j]) + (aH[1][0][j] + sg * aH[1][1][j]);
        out[0][h][zi][j] -= sgn * ti; out[1][h][zi][j] += sgn * tr;                 // (+-i) (tr + i ti)
      }
  }
#pragma unroll
  for (int h = 0; h < 2; ++h) {                                 // along the columns: D_y
    const int x = 8 * rb + 32 * h + g;
    double aG[2][2][2] = {}, aH[2][2][2] = {};
#pragma unroll
    for (int kb = 0; kb < 8; ++kb) {
      const int y1 = 4 * kb + t;
      const cplx w1 = T[oc_ix(0, x * 64 + y1, 1)], w2 = T[oc_ix(0, x * 64 + y1 + 32, 1)];
      const cplx h1 = cscale(w1, __ldg(Wy + x * 64 + y1)), h2 = cscale(w2, __ldg(Wy + x * 64 + y1 + 32));
      const double me = __ldg(my + 32 * kb), mo = __ldg(my + 1024 + 32 * kb);
      oc_dmma(aG[0][0][0], aG[0][0][1], w1.x + w2.x, me); oc_dmma(aG[0][1][0], aG[0][1][1], w1.x - w2.x, mo);
      oc_dmma(aG[1][0][0], aG[1][0][1], w1.y + w2.y, me); oc_dmma(aG[1][1][0], aG[1][1][1], w1.y - w2.y, mo);
      oc_dmma(aH[0][0][0], aH[0][0][1], h1.x + h2.x, me); oc_dmma(aH[0][1][0], aH[0][1][1], h1.x - h2.x, mo);
      oc_dmma(aH[1][0][0], aH[1][0][1], h1.y + h2.y, me); oc_dmma(aH[1][1][0], aH[1][1][1], h1.y - h2.y, mo);
    }
#pragma unroll
    for (int zi = 0; zi < 2; ++zi)
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const double sg = zi ? -1.0 : 1.0;
        const double wv = __ldg(Wy + x * 64 + 8 * cb + 32 * zi + 2 * t + j);
        const double tr = wv * (aG[0][0][j] + sg * aG[0][1][j]) + (aH[0][0][j] + sg * aH[0][1][j]);
        const double ti = wv * (aG[1][0][j] + sg * aG[1][1][j]) + (aH[1][0][j] + sg * aH[1][1][j]);
        out[0][h][zi][j] -= sgn * ti; out[1][h][zi][j] += sgn * tr;
      }
  }
}
__device__ __forceinline__ void oc_lap64_store(cplx* T, int rb, int cb, const double (&out)[2][2][2][2]) {
  const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
#pragma unroll
  for (int h = 0; h < 2; ++h)
#pragma unroll
    for (int zi = 0; zi < 2; ++zi)
#pragma unroll
      for (int j = 0; j < 2; ++j)
        T[oc_ix(0, (8 * rb + 32 * h + g) * 64 + 8 * cb + 32 * zi + 2 * t + j, 1)] = make_double2(out[0][h][zi][j], out[1][h][zi][j]);
}

// ---- lines of 128 points (quasi-1D, configs[1]): d^2 as the folded matrices Ce, Co (64 x 64) of Eq. 28b.  The batch is a
// matrix [lines][128]: the lines are the rows of the A operand, the matrices are the B operand.  Warp = (block of 8 lines, half
// of the folded columns), results in fragments until every warp has read its lines, then in place.
// Element i of line l is stored at oc_ix(l, i, 2).  The results stay in registers (res) until oc_lap128_store.
__device__ __forceinline__ void oc_lap128(const cplx* F, const double* mat, int lines, cplx (&res)[2][2][4]) {
  // two folds: e = w[k] + w[k+64], o = w[k] - w[k+64] (k < 64); the even part is again a symmetric circulant (period 64):
  // ee = e[k] + e[k+32], eo = e[k] - e[k+32] (k < 32).  O = Co o (64 x 64), EE = Cee ee, EO = Ceo eo (32 x 32);
  // E[i] = EE[i] + EO[i], E[i+32] = EE[i] - EO[i] (i < 32); out[i] = E[i] + O[i], out[i+64] = E[i] - O[i] (i < 64):
  // 6144 instead of 8192 multiply-adds per real line.  mat (fragment order, ctx.cuh): Co [8 blocks][16 kb][32],
  // then Cee, Ceo [4 blocks][8 kb][32] each.
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int lb = warp & 3, ch = warp >> 2, line = 8 * lb + g;
  const bool active = 8 * lb < lines;                           // (whole warp)
  const bool lv = line < lines;                                 // a ragged last batch: lines beyond it are neither read nor written
  const cplx* T = F + (lv ? line : 0) * 128;
  const int sw = (line & 1) << 2;
  double aO[4][2][2] = {}, aE[2][2][2][2] = {};                 // O: [b, b+1, b+4, b+5][re | im][j]; E: [b, b+1][EE | EO][re | im][j]
  const int b0 = 2 * ch;                                        // this warp's column blocks of the twice-folded part: b0, b0 + 1
  if (active) {
#pragma unroll 2
    for (int kb = 0; kb < 8; ++kb) {
      const int k1 = (4 * kb + t) ^ sw;
      const cplx w0 = T[k1], w1 = T[k1 + 32], w2 = T[k1 + 64], w3 = T[k1 + 96];   // (a line beyond the batch reads line 0: its results are dropped)
      const cplx e0 = cadd(w0, w2), e1 = cadd(w1, w3), o0 = csub(w0, w2), o1 = csub(w1, w3);   // e[k], e[k+32], o[k], o[k+32]
      const cplx ee = cadd(e0, e1), eo = csub(e0, e1);
#pragma unroll
      for (int q = 0; q < 4; ++q) {                             // O part: column blocks b0, b0 + 1, b0 + 4, b0 + 5; k-blocks kb and kb + 8
        const int cbb = b0 + (q & 1) + 4 * (q >> 1);
        const double m0 = __ldg(mat + (cbb * 16 + kb) * 32 + lane), m1 = __ldg(mat + (cbb * 16 + kb + 8) * 32 + lane);
        oc_dmma(aO[q][0][0], aO[q][0][1], o0.x, m0); oc_dmma(aO[q][1][0], aO[q][1][1], o0.y, m0);
        oc_dmma(aO[q][0][0], aO[q][0][1], o1.x, m1); oc_dmma(aO[q][1][0], aO[q][1][1], o1.y, m1);
      }
#pragma unroll
      for (int q = 0; q < 2; ++q) {                             // EE, EO: column blocks b0, b0 + 1 of 4; k-block kb of 8
        const double mee = __ldg(mat + 4096 + ((b0 + q) * 8 + kb) * 32 + lane), meo = __ldg(mat + 5120 + ((b0 + q) * 8 + kb) * 32 + lane);
        oc_dmma(aE[q][0][0][0], aE[q][0][0][1], ee.x, mee); oc_dmma(aE[q][0][1][0], aE[q][0][1][1], ee.y, mee);
        oc_dmma(aE[q][1][0][0], aE[q][1][0][1], eo.x, meo); oc_dmma(aE[q][1][1][0], aE[q][1][1][1], eo.y, meo);
      }
    }
  }
  // results of this thread: points i, i + 32, i + 64, i + 96 for (q, j), i = 8 (b0 + q) + 2 t + j
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const cplx EE = make_double2(aE[q][0][0][j], aE[q][0][1][j]), EO = make_double2(aE[q][1][0][j], aE[q][1][1][j]);
      const cplx Elo = cadd(EE, EO), Ehi = csub(EE, EO);       // E[i], E[i + 32]
      const cplx Olo = make_double2(aO[q][0][j], aO[q][1][j]), Ohi = make_double2(aO[q + 2][0][j], aO[q + 2][1][j]);   // O[i], O[i + 32]
      res[q][j][0] = cadd(Elo, Olo); res[q][j][2] = csub(Elo, Olo);
      res[q][j][1] = cadd(Ehi, Ohi); res[q][j][3] = csub(Ehi, Ohi);
    }
}

// The current / velocity coupling on lines of 128 points (one held axis): res += rot [ W (D w) + D (W w) ], D the first
// derivative as a circulant folded once (De, Do 64 x 64, fragment order at mat1), W_sigma [128] in global memory;
// rot = +i on the lines of u (even), -i on the lines of v (odd).  One column-block pair (q) at a time: 16 accumulators.
__device__ __forceinline__ void oc_cur128(const cplx* F, const double* mat1, const double* curW, int lines, cplx (&res)[2][2][4]) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int lb = warp & 3, ch = warp >> 2, line = 8 * lb + g;
  if (8 * lb >= lines) return;                                  // (whole warp)
  const bool lv = line < lines;
  const cplx* T = F + (lv ? line : 0) * 128;
  const int sw = (line & 1) << 2, b0 = 2 * ch;
  const double* W = curW + (line & 1) * 3 * 128;                // W_a | W_b along the held axis (M = 128)
  const double sgn = (line & 1) ? -1.0 : 1.0;
#pragma unroll 1
  for (int q = 0; q < 2; ++q) {
    double aG[2][2][2][2] = {}, aH[2][2][2][2] = {};            // [columns i | i + 32][re | im][E | O][j]
#pragma unroll 2
    for (int kb = 0; kb < 16; ++kb) {
      const int k = 4 * kb + t, k1 = k ^ sw;
      const cplx w1 = T[k1], w2 = T[k1 + 64];
      const cplx h1 = cscale(w1, __ldg(W + k)), h2 = cscale(w2, __ldg(W + k + 64));
      const cplx ew = cadd(w1, w2), ow = csub(w1, w2), eh = cadd(h1, h2), oh = csub(h1, h2);
#pragma unroll
      for (int hi = 0; hi < 2; ++hi) {
        const int cbb = b0 + q + 4 * hi;
        const double me = __ldg(mat1 + (cbb * 16 + kb) * 32 + lane), mo = __ldg(mat1 + 4096 + (cbb * 16 + kb) * 32 + lane);
        oc_dmma(aG[hi][0][0][0], aG[hi][0][0][1], ew.x, me); oc_dmma(aG[hi][0][1][0], aG[hi][0][1][1], ow.x, mo);
        oc_dmma(aG[hi][1][0][0], aG[hi][1][0][1], ew.y, me); oc_dmma(aG[hi][1][1][0], aG[hi][1][1][1], ow.y, mo);
        oc_dmma(aH[hi][0][0][0], aH[hi][0][0][1], eh.x, me); oc_dmma(aH[hi][0][1][0], aH[hi][0][1][1], oh.x, mo);
        oc_dmma(aH[hi][1][0][0], aH[hi][1][0][1], eh.y, me); oc_dmma(aH[hi][1][1][0], aH[hi][1][1][1], oh.y, mo);
      }
    }
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
      for (int p = 0; p < 4; ++p) {                             // point i + 32 p: columns block hi = p & 1, E + O (p < 2) or E - O
        const int hi = p & 1, i = 8 * (b0 + q) + 2 * t + j + 32 * p;
        const double sg = p < 2 ? 1.0 : -1.0, wv = __ldg(W + i);
        const double tr = wv * (aG[hi][0][0][j] + sg * aG[hi][0][1][j]) + (aH[hi][0][0][j] + sg * aH[hi][0][1][j]);
        const double ti = wv * (aG[hi][1][0][j] + sg * aG[hi][1][1][j]) + (aH[hi][1][0][j] + sg * aH[hi][1][1][j]);
        res[q][j][p].x -= sgn * ti; res[q][j][p].y += sgn * tr;
      }
  }
}

// overwrite the lines in place (after every warp has read them: the caller's barrier)
__device__ __forceinline__ void oc_lap128_store(cplx* F, int lines, const cplx (&res)[2][2][4]) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int lb = warp & 3, ch = warp >> 2, line = 8 * lb + g;
  if (8 * lb >= lines || line >= lines) return;
  cplx* W = F + line * 128;
  const int sw = (line & 1) << 2, b0 = 2 * ch;
#pragma unroll
  for (int q = 0; q < 2; ++q)
#pragma unroll
    for (int j = 0; j < 2; ++j) {
      const int i = (8 * (b0 + q) + 2 * t + j) ^ sw;
#pragma unroll
      for (int p = 0; p < 4; ++p) W[i + 32 * p] = res[q][j][p];
    }
}

// the same products with the results written in place from the accumulators (contains its two barriers): the variant
// without the coupling, which needs no result registers beside them
__device__ __forceinline__ void oc_lap128_inplace(cplx* F, const double* mat, int lines) {
  // two folds: e = w[k] + w[k+64], o = w[k] - w[k+64] (k < 64); the even part is again a symmetric circulant (period 64):
  // ee = e[k] + e[k+32], eo = e[k] - e[k+32] (k < 32).  O = Co o (64 x 64), EE = Cee ee, EO = Ceo eo (32 x 32);
  // E[i] = EE[i] + EO[i], E[i+32] = EE[i] - EO[i] (i < 32); out[i] = E[i] + O[i], out[i+64] = E[i] - O[i] (i < 64):
  // 6144 instead of 8192 multiply-adds per real line.  mat (fragment order, ctx.cuh): Co [8 blocks][16 kb][32],
  // then Cee, Ceo [4 blocks][8 kb][32] each.
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
  const int lb = warp & 3, ch = warp >> 2, line = 8 * lb + g;
  const bool active = 8 * lb < lines;                           // (whole warp)
  const bool lv = line < lines;                                 // a ragged last batch: lines beyond it are neither read nor written
  const cplx* T = F + (lv ? line : 0) * 128;
  const int sw = (line & 1) << 2;
  double aO[4][2][2] = {}, aE[2][2][2][2] = {};                 // O: [b, b+1, b+4, b+5][re | im][j]; E: [b, b+1][EE | EO][re | im][j]
  const int b0 = 2 * ch;                                        // this warp's column blocks of the twice-folded part: b0, b0 + 1
  if (active) {
#pragma unroll 2
    for (int kb = 0; kb < 8; ++kb) {
      const int k1 = (4 * kb + t) ^ sw;
      const cplx w0 = T[k1], w1 = T[k1 + 32], w2 = T[k1 + 64], w3 = T[k1 + 96];   // (a line beyond the batch reads line 0: its results are dropped)
      const cplx e0 = cadd(w0, w2), e1 = cadd(w1, w3), o0 = csub(w0, w2), o1 = csub(w1, w3);   // e[k], e[k+32], o[k], o[k+32]
      const cplx ee = cadd(e0, e1), eo = csub(e0, e1);
#pragma unroll
      for (int q = 0; q < 4; ++q) {                             // O part: column blocks b0, b0 + 1, b0 + 4, b0 + 5; k-blocks kb and kb + 8
        const int cbb = b0 + (q & 1) + 4 * (q >> 1);
        const double m0 = __ldg(mat + (cbb * 16 + kb) * 32 + lane), m1 = __ldg(mat + (cbb * 16 + kb + 8) * 32 + lane);
        oc_dmma(aO[q][0][0], aO[q][0][1], o0.x, m0); oc_dmma(aO[q][1][0], aO[q][1][1], o0.y, m0);
        oc_dmma(aO[q][0][0], aO[q][0][1], o1.x, m1); oc_dmma(aO[q][1][0], aO[q][1][1], o1.y, m1);
      }
#pragma unroll
      for (int q = 0; q < 2; ++q) {                             // EE, EO: column blocks b0, b0 + 1 of 4; k-block kb of 8
        const double mee = __ldg(mat + 4096 + ((b0 + q) * 8 + kb) * 32 + lane), meo = __ldg(mat + 5120 + ((b0 + q) * 8 + kb) * 32 + lane);
        oc_dmma(aE[q][0][0][0], aE[q][0][0][1], ee.x, mee); oc_dmma(aE[q][0][1][0], aE[q][0][1][1], ee.y, mee);
        oc_dmma(aE[q][1][0][0], aE[q][1][0][1], eo.x, meo); oc_dmma(aE[q][1][1][0], aE[q][1][1][1], eo.y, meo);
      }
    }
  }
  __syncthreads();
  if (active && lv) {
    cplx* W = F + line * 128;
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        const int i = (8 * (b0 + q) + 2 * t + j) ^ sw;            // i < 32
        const cplx EE = make_double2(aE[q][0][0][j], aE[q][0][1][j]), EO = make_double2(aE[q][1][0][j], aE[q][1][1][j]);
        const cplx Elo = cadd(EE, EO), Ehi = csub(EE, EO);       // E[i], E[i + 32]
        const cplx Olo = make_double2(aO[q][0][j], aO[q][1][j]), Ohi = make_double2(aO[q + 2][0][j], aO[q + 2][1][j]);   // O[i], O[i + 32]
        W[i] = cadd(Elo, Olo); W[i + 64] = csub(Elo, Olo);
        W[i + 32] = cadd(Ehi, Ohi); W[i + 96] = csub(Ehi, Ohi);
      }
  }
  __syncthreads();
}

template <int MODE, int MAXPT, int DM = 0, bool CUR = false>
__global__ void __launch_bounds__(MAXPT <= 2 ? 256 : 512, MAXPT <= 2 ? 2 : 1) k_onchip_stage(OCArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Lat& L = a.L;
  // the 64 x 64 matrix-form kernel (DM) is one spinor of 4096 points per batch on 512 threads: compile-time slot geometry
  const int lgM = DM == 1 ? 12 : DM == 2 ? 7 : L.lg[0] + L.lg[1] + L.lg[2], M = 1 << lgM, S = DM == 1 ? 1 : a.S, tid = threadIdx.x;
  const int NT = DM == 1 ? 512 : DM == 2 ? 256 : blockDim.x;
  cplx* F = reinterpret_cast<cplx*>(smem_raw);                       // [S][2][M]
  double* E = reinterpret_cast<double*>(F + (size_t)S * 2 * M);       // [S][M]
  __shared__ double s_eps[OC_MAXS], s_sn[OC_MAXS], s_red[16];
  // slots of this thread: lattice points i(kk) = (tid + 256 kk) & (M - 1), kk < PT; spinors s0, s0 + SSTEP, ...
  const int PT = DM == 1 ? 8 : DM == 2 ? 1 : M >= NT ? M / NT : 1;
  const int SSTEP = DM == 1 ? 1 : DM == 2 ? 2 : M >= NT ? 1 : NT / M, s0 = DM == 1 ? 0 : DM == 2 ? tid >> 7 : M >= NT ? 0 : tid >> lgM;
  // 4096 points (DM = 1): the 64 registers of per-thread density accumulators do not fit beside the spinor values (the
  // corrector spilled 488 bytes per thread): the densities of phi_new are taken by one streaming pass afterwards (oc_launch)
  constexpr bool NODENS = DM == 1;
  double acc[NODENS ? 1 : MAXPT][4];
#pragma unroll
  for (int kk = 0; kk < (NODENS ? 1 : MAXPT); ++kk) { acc[kk][0] = acc[kk][1] = acc[kk][2] = acc[kk][3] = 0.0; }
  // work slots of this thread: w -> (kk = w % PT, s = s0 + (w / PT) * SSTEP), at most OC_SLOTS of them; the spinor
  // values of the slots stay in registers from the load to the last phase (psi is read from HBM exactly once)
  const int nsp_full = DM == 1 ? 1 : S > s0 ? (S - s0 + SSTEP - 1) / SSTEP : 0;
  const int64_t n_batches = (a.n + S - 1) / S;
  for (int64_t b = blockIdx.x; b < n_batches; b += gridDim.x) {
    const int64_t n0 = b * S;
    const int cnt = (int)((a.n - n0 < S) ? a.n - n0 : S);
    const int used = cnt * 2 * M;
    const cplx* src = a.psi + (size_t)n0 * 2 * M;
    cplx ru[OC_SLOTS], rv[OC_SLOTS];
#pragma unroll
    for (int w = 0; w < OC_SLOTS; ++w) {
      ru[w] = rv[w] = make_double2(0.0, 0.0);
      if (w < PT * nsp_full) {
        const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
        if (sp < cnt) { ru[w] = __ldg(src + (size_t)(2 * sp) * M + i); rv[w] = __ldg(src + (size_t)(2 * sp + 1) * M + i); }
      }
    }
#pragma unroll
    for (int w = 0; w < OC_SLOTS; ++w) {
      if (w < PT * nsp_full) {
        const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
        if (a.scale && sp < cnt) { const double sc = a.scale[n0 + sp]; ru[w] = cscale(ru[w], sc); rv[w] = cscale(rv[w], sc); }
        F[(2 * sp) * M + oc_ix(0, i, DM)] = ru[w]; F[(2 * sp + 1) * M + oc_ix(1, i, DM)] = rv[w];
      }
    }
    __syncthreads();
    if (DM == 2) {                                              // lines of 128 points, 256 threads: d^2 in matrix form on DMMA
      if (CUR) {
        cplx res[2][2][4];
#pragma unroll
        for (int i = 0; i < 16; ++i) (&res[0][0][0])[i] = make_double2(0.0, 0.0);
        oc_lap128(F, a.mat, 2 * cnt, res);
        oc_cur128(F, a.mat + 6144, a.curW, 2 * cnt, res);
        __syncthreads();
        oc_lap128_store(F, 2 * cnt, res);
        __syncthreads();
      } else {
        oc_lap128_inplace(F, a.mat, 2 * cnt);
      }
      // the spinor values are read again (L2) instead of being held in registers across the matrix products
#pragma unroll
      for (int w = 0; w < OC_SLOTS; ++w) {
        ru[w] = rv[w] = make_double2(0.0, 0.0);
        if (w < PT * nsp_full) {
          const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
          if (sp < cnt) {
            const double sc = a.scale ? a.scale[n0 + sp] : 1.0;
            ru[w] = cscale(__ldcg(src + (size_t)(2 * sp) * M + i), sc); rv[w] = cscale(__ldcg(src + (size_t)(2 * sp + 1) * M + i), sc);
          }
        }
      }
      __syncthreads();
    } else if (DM == 1) {                                       // 64 x 64, 512 threads: lap u, lap v in place, matrix form on DMMA
      const int wp = tid >> 5, rb = wp & 3, cb = wp >> 2;
      for (int q = 0; q < 2 * cnt; ++q) {
        double lap[2][2][2][2];
        oc_lap64(F + (size_t)q * M, a.mat, rb, cb, lap);
        if (CUR) {                                              // lap - 2 (+-) cur(w): the stage's K = -1/2 (.) then carries the coupling
          const double* W = a.curW + (size_t)(q & 1) * 3 * M;
          oc_cur64(F + (size_t)q * M, a.mat + 4096, W, W + M, rb, cb, (q & 1) ? -1.0 : 1.0, lap);
        }
        __syncthreads();
        oc_lap64_store(F + (size_t)q * M, rb, cb, lap);
      }
      // the spinor values are read again (L2) instead of being held in 64 registers across the matrix products
#pragma unroll
      for (int w = 0; w < OC_SLOTS; ++w) {
        ru[w] = rv[w] = make_double2(0.0, 0.0);                 // (dead across the products on every path)
        if (w < PT * nsp_full) {
          const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
          if (sp < cnt) {
            const double sc = a.scale ? a.scale[n0 + sp] : 1.0;
            ru[w] = cscale(__ldcg(src + (size_t)(2 * sp) * M + i), sc); rv[w] = cscale(__ldcg(src + (size_t)(2 * sp + 1) * M + i), sc);
          }
        }
      }
      __syncthreads();
    } else {
      const int G = 2 * S;
      if (L.nd > 2) fft_axis<false>(F, G << (L.lg[0] + L.lg[1]), L.lg[2], 0, L.tw[2]);
      if (L.nd > 1) fft_axis<false>(F, G << L.lg[0], L.lg[1], L.lg[2], L.tw[1]);
      fft_axis<false>(F, G, L.lg[0], L.lg[1] + L.lg[2], L.tw[0]);
      for (int idx = tid; idx < used; idx += NT) {
        const int i = idx & (M - 1);
        const int j2 = i & (L.N[2] - 1), j1 = (i >> L.lg[2]) & (L.N[1] - 1), j0 = i >> (L.lg[1] + L.lg[2]);
        F[idx] = cscale(F[idx], kfactor(L, 0, j0, j1, j2).x);          // -k^2 / M at the stored (digit-reversed) position
      }
      __syncthreads();
      fft_axis<true>(F, G, L.lg[0], L.lg[1] + L.lg[2], L.tw[0]);
      if (L.nd > 1) fft_axis<true>(F, G << L.lg[0], L.lg[1], L.lg[2], L.tw[1]);
      if (L.nd > 2) fft_axis<true>(F, G << (L.lg[0] + L.lg[1]), L.lg[2], 0, L.tw[2]);
    }
    // ---- phase 1: H psi and the integrand of eps_n (F now holds lap u, lap v in natural order).  CORR leaves
    // X = C_part - i kappa H psi in F (phi_new = X + i kappa eps psi once eps_n is known): C_part is consumed here,
    // four slots at a time so that its loads are in flight together without holding 16 more values in registers.
    constexpr int WB = DM ? 2 : 4;                              // slots per batch of loads (4096 points: register budget)
#pragma unroll
    for (int w0 = 0; w0 < OC_SLOTS; w0 += WB) {
      cplx cu[WB], cv[WB];
      if (MODE == OC_CORR) {
#pragma unroll
        for (int r = 0; r < WB; ++r) {
          const int w = w0 + r;
          if (w < PT * nsp_full) {
            const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
            if (sp < cnt) { cu[r] = __ldg(a.cpart + (size_t)(2 * (n0 + sp)) * M + i); cv[r] = __ldg(a.cpart + (size_t)(2 * (n0 + sp) + 1) * M + i); }
          }
        }
      }
#pragma unroll
      for (int r = 0; r < WB; ++r) {
        const int w = w0 + r;
        if (w < PT * nsp_full) {
          const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
          if (sp < cnt) {
            const int64_t n = n0 + sp;
            const cplx D = cadd(a.F.delta[i], a.F.dext[i]);
            const double pa = a.F.U_a[i] - a.F.mu_a, pb = a.F.U_b[i] - a.F.mu_b, kp2 = a.kperp2[n];
            const cplx u = ru[w], v = rv[w];
            const int is = oc_ix(0, i, DM), it = oc_ix(1, i, DM);
            const cplx lu = F[(2 * sp) * M + is], lv = F[(2 * sp + 1) * M + it];
            const cplx Ku = make_double2(-0.5 * lu.x + 0.5 * kp2 * u.x, -0.5 * lu.y + 0.5 * kp2 * u.y);   // Eq. 14
            const cplx Kv = make_double2(-0.5 * lv.x + 0.5 * kp2 * v.x, -0.5 * lv.y + 0.5 * kp2 * v.y);
            const cplx Hu = cadd(Ku, cadd(cscale(u, pa), cmul(D, v)));                                    // Eqs. 5, 15
            const cplx Hv = csub(cmul(cconj(D), u), cadd(Kv, cscale(v, pb)));
            E[(sp << lgM) + i] = u.x * Hu.x + u.y * Hu.y + v.x * Hv.x + v.y * Hv.y;
            if (MODE == OC_APPLY) {
              a.out[(size_t)(2 * n) * M + i] = Hu; a.out[(size_t)(2 * n + 1) * M + i] = Hv;
            } else if (MODE == OC_RHS) {
              F[(2 * sp) * M + is] = Hu; F[(2 * sp + 1) * M + it] = Hv;
            } else {
              F[(2 * sp) * M + is] = make_double2(cu[r].x + a.kappa * Hu.y, cu[r].y - a.kappa * Hu.x);
              F[(2 * sp + 1) * M + it] = make_double2(cv[r].x + a.kappa * Hv.y, cv[r].y - a.kappa * Hv.x);
            }
          }
        }
      }
    }
    __syncthreads();
    if (DM == 1) oc_reduce1(E, s_red, s_eps); else oc_reduce(E, cnt, lgM, s_eps);
    __syncthreads();
    if (tid < cnt) {
      const double e_true = a.dV * s_eps[tid];
      if (a.eps_out) a.eps_out[n0 + tid] = e_true;
      s_eps[tid] = (a.use_shift && MODE != OC_APPLY) ? e_true : 0.0;
    }
    __syncthreads();
    if (MODE != OC_APPLY) {
      // ---- phase 2: f = -i (H - eps) psi;  RHS writes it, CORR forms phi_new = C_part + kappa f in place
#pragma unroll
      for (int w = 0; w < OC_SLOTS; ++w) {
        if (w < PT * nsp_full) {
          const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
          if (sp < cnt) {
            const int64_t n = n0 + sp;
            const double e = s_eps[sp];
            const cplx u = ru[w], v = rv[w];
            const cplx Hu = F[(2 * sp) * M + oc_ix(0, i, DM)], Hv = F[(2 * sp + 1) * M + oc_ix(1, i, DM)];
            if (MODE == OC_RHS) {
              const cplx fu = make_double2(Hu.y - e * u.y, -(Hu.x - e * u.x)), fv = make_double2(Hv.y - e * v.y, -(Hv.x - e * v.x));
              a.out[(size_t)(2 * n) * M + i] = fu; a.out[(size_t)(2 * n + 1) * M + i] = fv;
            } else {
              const double ke = a.kappa * e;                           // F holds X: phi_new = X + i kappa eps psi
              const cplx pu = make_double2(Hu.x - ke * u.y, Hu.y + ke * u.x);
              const cplx pv = make_double2(Hv.x - ke * v.y, Hv.y + ke * v.x);
              ru[w] = pu; rv[w] = pv;                                  // phi_new stays in registers
              E[(sp << lgM) + i] = cabs2(pu) + cabs2(pv);
            }
          }
        }
      }
    }
    if (MODE == OC_CORR) {
      __syncthreads();
      if (DM == 1) oc_reduce1(E, s_red, s_sn); else oc_reduce(E, cnt, lgM, s_sn);
      __syncthreads();
      if (tid < cnt) s_sn[tid] = a.normalize ? 1.0 / sqrt(a.dV * s_sn[tid]) : 1.0;
      __syncthreads();
      // ---- phase 3: normalise (Alg. 2 step 8), write phi_new once, accumulate its densities (Eqs. 7a, 7b, 7e)
#pragma unroll
      for (int w = 0; w < OC_SLOTS; ++w) {
        if (w < PT * nsp_full) {
          const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
          if (sp < cnt) {
            const int64_t n = n0 + sp;
            const double sn = s_sn[sp];
            const cplx u = cscale(ru[w], sn), v = cscale(rv[w], sn);
            a.out[(size_t)(2 * n) * M + i] = u; a.out[(size_t)(2 * n + 1) * M + i] = v;
            if (!NODENS && a.do_dens) {
              const double cp = a.cpref[n], wa = a.w_a[n], wb = a.w_b[n], wn = 0.5 * cp * (wb - wa);
              oc_dens_acc<(NODENS ? 1 : MAXPT)>(acc, w, PT, cp * wa * cabs2(u), cp * wb * cabs2(v), wn * (u.x * v.x + u.y * v.y), wn * (u.y * v.x - u.x * v.y));
            }
          }
        }
      }
    }
    __syncthreads();
  }
  if (!NODENS && MODE == OC_CORR && a.do_dens) {
    const int slots = PT * NT;
    double* dp = a.dpart + (size_t)blockIdx.x * 4 * slots;
#pragma unroll
    for (int kk = 0; kk < (NODENS ? 1 : MAXPT); ++kk)
      if (kk < PT)
#pragma unroll
        for (int f = 0; f < 4; ++f) dp[f * slots + tid + NT * kk] = acc[kk][f];
  }
}

// Alg. 2 steps 1-2 on chip: P = phi + dt sum b_i f_i and C_part = phi + dt sum_{i>=1} c_i f_i in one
// sweep over phi and the history, |P| reduced inside the CTA, the NORMALISED predictor written over phi, C_part over
// the oldest history buffer, and the densities of the predictor accumulated per CTA: 5 reads + 2 writes, nothing else.
struct OCPred {
  Lat L;
  cplx* phi; HistPtrs h; cplx* cpart; AbmCoef k;
  double dV; int normalize;
  int do_dens; const double *cpref, *w_a, *w_b; double* dpart;
  int64_t n; int S;
};

template <int MAXPT>
__global__ void __launch_bounds__(MAXPT <= 2 ? 256 : 512, MAXPT <= 2 ? 2 : 1) k_onchip_pred(OCPred a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Lat& L = a.L;
  const int lgM = L.lg[0] + L.lg[1] + L.lg[2], M = 1 << lgM, S = a.S, tid = threadIdx.x, NT = blockDim.x;
  cplx* F = reinterpret_cast<cplx*>(smem_raw);
  double* E = reinterpret_cast<double*>(F + (size_t)S * 2 * M);
  __shared__ double s_sn[OC_MAXS], s_red[16];
  const int PT = M >= NT ? M / NT : 1;
  const int SSTEP = M >= NT ? 1 : NT / M, s0 = M >= NT ? 0 : tid >> lgM;
  double acc[MAXPT][4];
#pragma unroll
  for (int kk = 0; kk < MAXPT; ++kk) { acc[kk][0] = acc[kk][1] = acc[kk][2] = acc[kk][3] = 0.0; }
  const int64_t n_batches = (a.n + S - 1) / S;
  for (int64_t b = blockIdx.x; b < n_batches; b += gridDim.x) {
    const int64_t n0 = b * S;
    const int cnt = (int)((a.n - n0 < S) ? a.n - n0 : S);
    // work slots of this thread: w -> (kk = w % PT, s = s0 + (w / PT) * SSTEP); two slots per round so that 2 x 2 x (1 + m)
    // independent 16-byte loads are in flight before the first use
    const int nsp = cnt > s0 ? (cnt - s0 + SSTEP - 1) / SSTEP : 0, W = PT * nsp;
    constexpr int R = MAXPT <= 2 ? 2 : 1;                      // slots per round (MAXPT = 8: 64 registers hold the density accumulators)
    for (int w0 = 0; w0 < W; w0 += R) {
      cplx ph[R][2], fh[R][2][5];
      size_t off[R][2];
      int si[R], ii[R];
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const int w = w0 + r < W ? w0 + r : W - 1;               // the tail repeats the last slot (harmless: same values)
        ii[r] = (tid + NT * (w % PT)) & (M - 1); si[r] = s0 + (w / PT) * SSTEP;
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
          off[r][cc] = (size_t)(2 * (n0 + si[r]) + cc) * M + ii[r];
          ph[r][cc] = __ldg(a.phi + off[r][cc]);
#pragma unroll
          for (int j = 0; j < 5; ++j)
            if (j < a.k.ab || j + 1 < a.k.am) fh[r][cc][j] = __ldg(a.h.f[j] + off[r][cc]);
        }
      }
#pragma unroll
      for (int r = 0; r < R; ++r) {
        if (w0 + r >= W) break;
        double nrm = 0.0;
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
          cplx p = ph[r][cc], q = p;
#pragma unroll
          for (int j = 0; j < 5; ++j) {
            if (j < a.k.ab) { p.x += a.k.b[j] * fh[r][cc][j].x; p.y += a.k.b[j] * fh[r][cc][j].y; }
            if (j + 1 < a.k.am) { q.x += a.k.c[j + 1] * fh[r][cc][j].x; q.y += a.k.c[j + 1] * fh[r][cc][j].y; }
          }
          a.cpart[off[r][cc]] = q;
          F[(2 * si[r] + cc) * M + ii[r]] = p;
          nrm += cabs2(p);
        }
        E[(si[r] << lgM) + ii[r]] = nrm;
      }
    }
    __syncthreads();
    if (M == 4096 && NT == 512) oc_reduce1(E, s_red, s_sn); else oc_reduce(E, cnt, lgM, s_sn);     // S = 1: all 16 warps
    __syncthreads();
    if (tid < cnt) s_sn[tid] = a.normalize ? 1.0 / sqrt(a.dV * s_sn[tid]) : 1.0;
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < MAXPT; ++kk) {
      if (kk < PT) {
        const int i = (tid + NT * kk) & (M - 1);
        for (int s = s0; s < cnt; s += SSTEP) {
          const int64_t n = n0 + s;
          const double sn = s_sn[s];
          const cplx u = cscale(F[(2 * s) * M + i], sn), v = cscale(F[(2 * s + 1) * M + i], sn);
          a.phi[(size_t)(2 * n) * M + i] = u; a.phi[(size_t)(2 * n + 1) * M + i] = v;
          if (a.do_dens) {
            const double cp = a.cpref[n], wa = a.w_a[n], wb = a.w_b[n], wn = 0.5 * cp * (wb - wa);
            acc[kk][0] += cp * wa * cabs2(u);
            acc[kk][1] += cp * wb * cabs2(v);
            acc[kk][2] += wn * (u.x * v.x + u.y * v.y);
            acc[kk][3] += wn * (u.y * v.x - u.x * v.y);
          }
        }
      }
    }
    __syncthreads();
  }
  if (a.do_dens) {
    const int slots = PT * NT;
    double* dp = a.dpart + (size_t)blockIdx.x * 4 * slots;
#pragma unroll
    for (int kk = 0; kk < MAXPT; ++kk)
      if (kk < PT)
#pragma unroll
        for (int f = 0; f < 4; ++f) dp[f * slots + tid + NT * kk] = acc[kk][f];
  }
}

// raw[f][i] = sum over CTAs and duplicate slots of a lattice point, in a fixed order (one warp per output)
__global__ void k_oc_dens_final(const double* dpart, int n_cta, int slots, int64_t M, double* raw) {
  const int64_t o = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (o >= 4 * M) return;
  const int f = (int)(o / M); const int64_t i = o - f * M;
  const int dup = (int)(slots / M), terms = n_cta * dup;
  double s = 0.0;
  for (int t = lane; t < terms; t += 32) {
    const int cta = t / dup, d = t - cta * dup;
    s += dpart[((size_t)cta * 4 + f) * slots + i + (int64_t)d * M];
  }
  for (int k = 16; k > 0; k >>= 1) s += __shfl_xor_sync(0xffffffffu, s, k);
  if (lane == 0) raw[o] = s;
}

// ---- host side ------------------------------------------------------------------------------------------------
static bool g_oc_attr_done = false;
static void oc_launch(wslda_ctx* c, cudaStream_t st, int mode, const cplx* psi, const double* scale, int64_t n0, int64_t n,
                      cplx* out, const cplx* cpart, double kappa, int do_dens, double* eps_user) {
  const Plan& P = c->P;
  OCArgs a;
  a.L = c->L; a.psi = psi; a.scale = scale; a.kperp2 = c->kperp2 + n0; a.F = fields_of(c);
  a.out = out; a.cpart = cpart; a.kappa = kappa; a.dV = c->dV;
  a.use_shift = c->f.subtract_mean_energy; a.normalize = c->f.normalize; a.eps_out = eps_user;
  a.do_dens = do_dens; a.cpref = c->cpref + n0; a.w_a = c->w_a + n0; a.w_b = c->w_b + n0; a.dpart = c->oc_dpart;
  a.n = n; a.S = P.ocS; a.dm = c->oc_dm; a.mat = c->oc_mat; a.curW = (c->f.current_terms && c->oc_dm) ? c->cur_W : nullptr;
  const size_t smem = (size_t)P.ocS * 2 * P.M * 16 + (size_t)P.ocS * P.M * 8;
  if (!g_oc_attr_done) {
    cudaFuncSetAttribute(k_onchip_stage<OC_APPLY, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_CORR, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_RHS, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_APPLY, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_CORR, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_RHS, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_APPLY, 2, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_CORR, 2, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_RHS, 2, 2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_APPLY, 2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_CORR, 2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_RHS, 2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_APPLY, 8, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_CORR, 8, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_RHS, 8, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_APPLY, 8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_CORR, 8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_RHS, 8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    g_oc_attr_done = true;
  }
  const bool small = P.M <= 512;
  const int NT = small ? 256 : 512;
  const int64_t nbat = (n + P.ocS - 1) / P.ocS;
  const int grid = (int)(nbat < P.oc_grid ? nbat : P.oc_grid);
  const double lgM = (double)(P.lg[0] + P.lg[1] + P.lg[2]);
  WORK(c, 32.0 * P.M * n * (mode == OC_CORR ? 3.0 : 2.0), 5.0 * P.M * lgM * 2.0 * 2.0 * n);
  void (*k)(OCArgs);
  if (small && c->oc_dm == 2 && a.curW) k = mode == OC_APPLY ? k_onchip_stage<OC_APPLY, 2, 2, true> : mode == OC_CORR ? k_onchip_stage<OC_CORR, 2, 2, true> : k_onchip_stage<OC_RHS, 2, 2, true>;
  else if (small && c->oc_dm == 2) k = mode == OC_APPLY ? k_onchip_stage<OC_APPLY, 2, 2> : mode == OC_CORR ? k_onchip_stage<OC_CORR, 2, 2> : k_onchip_stage<OC_RHS, 2, 2>;
  else if (small) k = mode == OC_APPLY ? k_onchip_stage<OC_APPLY, 2> : mode == OC_CORR ? k_onchip_stage<OC_CORR, 2> : k_onchip_stage<OC_RHS, 2>;
  else if (c->oc_dm == 1 && a.curW) k = mode == OC_APPLY ? k_onchip_stage<OC_APPLY, 8, 1, true> : mode == OC_CORR ? k_onchip_stage<OC_CORR, 8, 1, true> : k_onchip_stage<OC_RHS, 8, 1, true>;
  else if (c->oc_dm == 1) k = mode == OC_APPLY ? k_onchip_stage<OC_APPLY, 8, 1> : mode == OC_CORR ? k_onchip_stage<OC_CORR, 8, 1> : k_onchip_stage<OC_RHS, 8, 1>;
  else k = mode == OC_APPLY ? k_onchip_stage<OC_APPLY, 8> : mode == OC_CORR ? k_onchip_stage<OC_CORR, 8> : k_onchip_stage<OC_RHS, 8>;
  LAUNCHN(c, mode == OC_APPLY ? "k_onchip_apply" : mode == OC_CORR ? "k_onchip_corr" : "k_onchip_rhs", k, grid, NT, smem, st, a);
  if (mode == OC_CORR && do_dens) {
    if (c->oc_dm == 1) {                                     // 64 x 64: one streaming pass over the normalised phi_new
      dens_chunk(c, out, nullptr, n0, n, WSLDA_D_RHO | WSLDA_D_NU, 0, st);
    } else {
      const int slots = (int)(P.M > NT ? P.M : NT);
      LAUNCH(c, k_oc_dens_final, nb(4 * P.M * 32, 256), 256, 0, st, c->oc_dpart, grid, slots, P.M, c->raw);
    }
  }
}

static wslda_status oc_apply_h(wslda_ctx* c, const cplx* psi, cplx* hpsi, double* eps_dev, int64_t n_first, int64_t n_count,
                               cudaStream_t st) {
  const int64_t M = c->P.M;
  if (n_count > 0)
    oc_launch(c, st, OC_APPLY, psi + 2 * n_first * M, nullptr, n_first, n_count, hpsi + 2 * n_first * M, nullptr, 0.0, 0,
              eps_dev ? eps_dev + n_first : c->eps + n_first);
  return cuda_check(c, "apply_h");
}

static void oc_pred(wslda_ctx* c, cudaStream_t st, cplx* phi, const HistPtrs& h, cplx* cpart, const AbmCoef& k, int do_dens) {
  const Plan& P = c->P;
  OCPred a;
  a.L = c->L; a.phi = phi; a.h = h; a.cpart = cpart; a.k = k; a.dV = c->dV; a.normalize = c->f.normalize;
  a.do_dens = do_dens; a.cpref = c->cpref; a.w_a = c->w_a; a.w_b = c->w_b; a.dpart = c->oc_dpart; a.n = P.n_wf; a.S = P.ocS;
  const size_t smem = (size_t)P.ocS * 2 * P.M * 16 + (size_t)P.ocS * P.M * 8;
  static bool attr = false;
  if (!attr) {
    cudaFuncSetAttribute(k_onchip_pred<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_pred<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    attr = true;
  }
  const bool small = P.M <= 512;
  const int NT = small ? 256 : 512;
  const int64_t nbat = (P.n_wf + P.ocS - 1) / P.ocS;
  const int grid = (int)(nbat < P.oc_grid ? nbat : P.oc_grid);
  WORK(c, 32.0 * P.M * P.n_wf * (1 + c->m + 2), 0);
  if (small) LAUNCHN(c, "k_onchip_pred", k_onchip_pred<2>, grid, NT, smem, st, a);
  else LAUNCHN(c, "k_onchip_pred", k_onchip_pred<8>, grid, NT, smem, st, a);
  if (do_dens) {
    const int slots = (int)(P.M > NT ? P.M : NT);
    LAUNCH(c, k_oc_dens_final, nb(4 * P.M * 32, 256), 256, 0, st, c->oc_dpart, grid, slots, P.M, c->raw);
  }
}
