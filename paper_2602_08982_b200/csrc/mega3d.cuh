// mega3d.cuh -- one persistent dataflow kernel per ABM stage for the fused 3-D path (Ny = Nz = 32).
//
// The three transform passes of fast3d.cuh and the stage epilogue become four kinds of work items over groups
// of `gs` spinors, handed out in ONE order by an atomic ticket counter to resident CTAs of 4 warps:
//   tick t :  A(t)   planes forward        -> spec ring slot t % R
//             B(t-1) x-lines, -k^2/M       (in place)
//             C(t-2) planes inverse + BdG mix + ABM combination -> X ring slot / H psi, partial sums
//             D(t-3) per-spinor scalars (eps_n, norm), final combination, densities
// An item waits (one thread spins on a completion counter in L2) only for items handed out EARLIER, which are
// being processed by running CTAs, so the scheme cannot deadlock whatever the residency; spins are bounded and
// raise an error flag.  All kinds are resident on every SM at the same time, so HBM-bound (A load, C/D
// epilogue), L2-bound (spectra) and FP64-bound (butterflies) phases overlap, and the spectra of only ~3 groups
// are live: they never leave the 126 MB L2.  Scratch written by other CTAs is read with ld.global.cg.
#pragma once
#include "fast3d.cuh"

#define F3_RING 4
#define F3_DSPLIT 2            // D items per x-plane

struct F3Sync {                // device counters, zeroed before every launch
  int next;                    // ticket
  int error;                   // set when a bounded spin ran out
  int pad[2];
  // followed by done[4][G] ints
};

struct F3Mega {
  const cplx* psi;             // [n][2][M]  input spinors (P or phi), first spinor of the call
  const double* scale;         // per spinor (nullable)
  const double* kperp2;        // per spinor
  F3Fields F;
  const double *ky2, *kz2;
  double kx2[32];
  double invM, dV, kappa;
  cplx* spec0; cplx* spec1;    // rings [R][gs][2][M]
  cplx* X;                     // ring  [R][gs][2][M]   (CORR / RHS)
  cplx* out;                   // APPLY: H psi; CORR: phi_new (= psi buffer); RHS: f_new        [n][2][M]
  const cplx* cpart;           // CORR
  double* part;                // [F3_NPART][n * NX]
  double* eps_out;             // per spinor: eps_n (true value; APPLY writes it from k_f3_scal instead)
  int use_shift, normalize, do_dens;
  const double *cpref, *w_a, *w_b;   // densities
  double* acc;                 // ring [R][4][M]
  F3Sync* sync;
  int n, gs, G, NX;
};

__device__ __forceinline__ cplx ldcg2(const cplx* p) { return __ldcg(p); }

// one thread waits until *ctr >= target (bounded), then the whole CTA proceeds
__device__ __forceinline__ void f3_wait(int* ctr, int target, F3Sync* sy) {
  if (threadIdx.x == 0) {
    int spins = 0;
    while (*(volatile int*)ctr < target) {
      __nanosleep(200);
      if (++spins > (1 << 23)) { sy->error = 1; break; }
    }
    __threadfence();
  }
  __syncthreads();
}
__device__ __forceinline__ void f3_signal(int* ctr) {
  __syncthreads();
  if (threadIdx.x == 0) { __threadfence(); atomicAdd(ctr, 1); }
}

// ---- A: forward plane transforms of 4 component planes (one per warp) ----------------------------------------
template <bool SYM>
__device__ __forceinline__ void f3_body_a(const F3Mega& a, int g, int ia, cplx* tiles, cplx* x) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int p = 4 * ia + warp, nl = p / (2 * a.NX), rem = p - nl * 2 * a.NX, c = rem / a.NX, ix = rem - c * a.NX;
  const int n = g * a.gs + nl;
  if (n >= a.n) return;
  cplx* S = tiles + warp * (F3_N * F3_PITCH);
  const size_t M = (size_t)a.NX * F3_PLANE;
  const cplx* src = a.psi + ((size_t)(2 * n + c) * a.NX + ix) * F3_PLANE;
  const double s = a.scale ? a.scale[n] : 1.0;
  const double* al = a.F.alpha[c] + (size_t)ix * F3_PLANE;
  const size_t sb = (((size_t)(g % F3_RING) * a.gs + nl) * 2 + c) * M + (size_t)ix * F3_PLANE;
#pragma unroll 1
  for (int t = 0; t < (SYM ? 2 : 1); ++t) {
#pragma unroll
    for (int j = 0; j < F3_N; ++j) {
      double f = s;
      if (SYM && t) f *= al[j * F3_N + lane];
      x[j] = cscale(src[j * F3_N + lane], f);
    }
    f3_plane_forward(x, S, lane);
    cplx* dst = (t == 0 ? a.spec0 : a.spec1) + sb;
#pragma unroll
    for (int j = 0; j < F3_N; ++j) dst[j * F3_N + lane] = x[j];
  }
}

// ---- B: x-lines of 4 (component, kz) rows: FFT x, -k^2/M, inverse FFT x, in place ------------------------------
template <int NX, bool SYM>
__device__ __forceinline__ void f3_body_b(const F3Mega& a, int g, int ib, cplx* x) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q = 4 * ib + warp, kz = q & (F3_N - 1), ccl = q >> 5;
  if (g * a.gs + (ccl >> 1) >= a.n) return;
  const size_t M = (size_t)NX * F3_PLANE;
  const double kyz2 = a.ky2[lane] + a.kz2[kz];
  const size_t sb = ((size_t)(g % F3_RING) * a.gs * 2 + ccl) * M + kz * F3_N + lane;
#pragma unroll 1
  for (int t = 0; t < (SYM ? 2 : 1); ++t) {
    cplx* p = (t ? a.spec1 : a.spec0) + sb;
#pragma unroll
    for (int j = 0; j < NX; ++j) x[j] = ldcg2(p + (size_t)j * F3_PLANE);
#pragma unroll 1
    for (int dir = 0; dir < 2; ++dir) {
      fft_reg<NX, false>(x);
#pragma unroll
      for (int j = 0; j < NX; ++j) {
        const double f = dir ? 1.0 : -(a.kx2[j] + kyz2) * a.invM;
        x[j] = make_double2(x[j].x * f, -x[j].y * f);
      }
    }
#pragma unroll
    for (int j = 0; j < NX; ++j) p[(size_t)j * F3_PLANE] = x[j];
  }
}

// ---- C: inverse plane transforms (one per warp), then the pointwise BdG mix and the stage combination ----------
// SYM: the 4 warps hold alpha lap u | lap(alpha u) | alpha lap v | lap(alpha v) of ONE (spinor, x-plane);
// Eq. 14: lap u | lap v of TWO x-planes.  Each warp leaves its plane in its own tile; after the barrier every
// thread finishes 32 / WPI rows of both components (psi, C_part and the fields are read once per point).
template <bool SYM, int MODE>
__device__ __forceinline__ void f3_body_c(const F3Mega& a, int g, int ic, cplx* tiles, double* red, cplx* x) {
  constexpr int NS = SYM ? 2 : 1, WPI = 2 * NS, IPC = 4 / WPI, ROWS = F3_N / WPI, TILE = F3_N * F3_PITCH;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int pI = warp / WPI, wl = warp % WPI, c = wl / NS, t = wl % NS;
  const int item = ic * IPC + pI, nl = item / a.NX, ix = item - nl * a.NX, n = g * a.gs + nl;
  const bool valid = n < a.n;
  const size_t M = (size_t)a.NX * F3_PLANE, pl = (size_t)ix * F3_PLANE;
  const size_t ring = ((size_t)(g % F3_RING) * a.gs + nl) * 2;        // ring index of component 0 of this spinor
  cplx* S = tiles + warp * TILE;
  if (valid) {
    const cplx* sp = (t ? a.spec1 : a.spec0) + (ring + c) * M + pl;
#pragma unroll
    for (int j = 0; j < F3_N; ++j) x[j] = cconj(ldcg2(sp + j * F3_N + lane));
    f3_plane_forward(x, S, lane);                                    // conj of the value at (y = j, z = lane)
    const double* al = a.F.alpha[c] + pl;
#pragma unroll
    for (int j = 0; j < F3_N; ++j) {
      const double f = (SYM && t == 0) ? al[j * F3_N + lane] : 1.0;
      S[j * F3_PITCH + lane] = make_double2(x[j].x * f, -x[j].y * f);
    }
  }
  __syncthreads();
  double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
  if (valid) {
    const cplx* tb = tiles + pI * WPI * TILE;
    const double s = a.scale ? a.scale[n] : 1.0, kp2 = a.kperp2[n];
    const cplx* pu = a.psi + (size_t)(2 * n) * M + pl;
    const cplx* pv = pu + M;
    cplx* ou = (MODE == F3_APPLY ? a.out + (size_t)(2 * n) * M : a.X + ring * M) + pl;
    cplx* ov = ou + M;
    const cplx* cu = a.cpart + (size_t)(2 * n) * M + pl;
#pragma unroll 4
    for (int jj = 0; jj < ROWS; ++jj) {
      const int j = wl * ROWS + jj, i = j * F3_N + lane, si = j * F3_PITCH + lane;
      const cplx u = cscale(pu[i], s), v = cscale(pv[i], s);
      const cplx Lu = tb[(NS - 1) * TILE + si], Lv = tb[(2 * NS - 1) * TILE + si];
      cplx Ku, Kv;
      if (SYM) {
        const cplx Tu = tb[si], Tv = tb[NS * TILE + si];
        const double aa = a.F.alpha[0][pl + i], ab = a.F.alpha[1][pl + i], la = a.F.lap[0][pl + i], lb = a.F.lap[1][pl + i];
        const double ha = 0.5 * aa * kp2, hb = 0.5 * ab * kp2;
        Ku.x = -0.25 * (Lu.x + Tu.x - la * u.x) + ha * u.x;            // Eq. 40 + transverse shift
        Ku.y = -0.25 * (Lu.y + Tu.y - la * u.y) + ha * u.y;
        Kv.x = -0.25 * (Lv.x + Tv.x - lb * v.x) + hb * v.x;
        Kv.y = -0.25 * (Lv.y + Tv.y - lb * v.y) + hb * v.y;
      } else {
        Ku = make_double2(-0.5 * Lu.x + 0.5 * kp2 * u.x, -0.5 * Lu.y + 0.5 * kp2 * u.y);     // Eq. 14
        Kv = make_double2(-0.5 * Lv.x + 0.5 * kp2 * v.x, -0.5 * Lv.y + 0.5 * kp2 * v.y);
      }
      const cplx D = cadd(a.F.delta[pl + i], a.F.dext[pl + i]);
      const double pa = a.F.U[0][pl + i] - a.F.mu[0], pb = a.F.U[1][pl + i] - a.F.mu[1];
      const cplx Hu = cadd(Ku, cadd(cscale(u, pa), cmul(D, v)));                                // Eqs. 5, 15
      const cplx Hv = csub(cmul(cconj(D), u), cadd(Kv, cscale(v, pb)));
      e += u.x * Hu.x + u.y * Hu.y + v.x * Hv.x + v.y * Hv.y;
      if (MODE == F3_APPLY) { ou[i] = Hu; ov[i] = Hv; }
      else if (MODE == F3_RHS) { ou[i] = make_double2(Hu.y, -Hu.x); ov[i] = make_double2(Hv.y, -Hv.x); }   // -i H
      else {
        const cplx c0 = cu[i], c1 = cu[M + i];
        const cplx xu = make_double2(c0.x + a.kappa * Hu.y, c0.y - a.kappa * Hu.x);             // C_part - i kappa H
        const cplx xv = make_double2(c1.x + a.kappa * Hv.y, c1.y - a.kappa * Hv.x);
        ou[i] = xu; ov[i] = xv;
        xx += cabs2(xu) + cabs2(xv);
        xpr += xu.x * u.x + xu.y * u.y + xv.x * v.x + xv.y * v.y;
        xpi += xu.x * u.y - xu.y * u.x + xv.x * v.y - xv.y * v.x;
        pp += cabs2(u) + cabs2(v);
      }
    }
  }
  e = warp_sum(e);
  if (MODE == F3_CORR) { xx = warp_sum(xx); xpr = warp_sum(xpr); xpi = warp_sum(xpi); pp = warp_sum(pp); }
  if (lane == 0) {
    red[warp * F3_NPART] = e;
    if (MODE == F3_CORR) { red[warp * F3_NPART + 1] = xx; red[warp * F3_NPART + 2] = xpr; red[warp * F3_NPART + 3] = xpi; red[warp * F3_NPART + 4] = pp; }
  }
  __syncthreads();
  if (valid && wl == 0 && lane == 0) {
    const size_t np = (size_t)a.n * a.NX;
    for (int k = 0; k < (MODE == F3_CORR ? F3_NPART : 1); ++k) {
      double sum = 0.0;
      for (int w = 0; w < WPI; ++w) sum += red[(pI * WPI + w) * F3_NPART + k];
      a.part[k * np + (size_t)n * a.NX + ix] = sum;
    }
  }
}

// ---- D: per-spinor scalars of the group, then the final combination of half an x-plane for every spinor ---------
// CORR: phi_new = (X + i kappa eps w) * scale_new over P (Alg. 2 steps 4, 8) + densities of phi_new;
// RHS : f_new = Y + i eps phi (Alg. 2 step 9, Eq. 45b).
template <int MODE>
__device__ __forceinline__ void f3_body_d(const F3Mega& a, int g, int id, double* s_eps, double* s_sn) {
  constexpr int PTS = F3_PLANE / F3_DSPLIT / 128;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int ix = id / F3_DSPLIT, half = id - ix * F3_DSPLIT;
  const int cnt = (a.n - g * a.gs < a.gs) ? a.n - g * a.gs : a.gs;
  const size_t M = (size_t)a.NX * F3_PLANE, np = (size_t)a.n * a.NX;
  for (int nl = warp; nl < cnt; nl += 4) {
    const int n = g * a.gs + nl;
    double v[F3_NPART];
#pragma unroll
    for (int k = 0; k < F3_NPART; ++k) {
      double t = 0.0;
      if ((k == 0 || MODE == F3_CORR) && lane < a.NX) t = __ldcg(a.part + k * np + (size_t)n * a.NX + lane);
      v[k] = warp_sum(t);
    }
    if (lane == 0) {
      const double e_true = a.dV * v[0], e = a.use_shift ? e_true : 0.0;
      s_eps[nl] = e;
      if (id == 0 && a.eps_out) a.eps_out[n] = e_true;
      if (MODE == F3_CORR) {
        const double ke = a.kappa * e, nrm2 = a.dV * (v[1] - 2.0 * ke * v[3] + ke * ke * v[4]);
        s_sn[nl] = a.normalize ? 1.0 / sqrt(nrm2) : 1.0;
      }
    }
  }
  __syncthreads();
  const size_t p0 = (size_t)ix * F3_PLANE + half * (F3_PLANE / F3_DSPLIT) + threadIdx.x;
  const size_t ring = (size_t)(g % F3_RING) * a.gs * 2;
  double acc[PTS][4];
#pragma unroll
  for (int r = 0; r < PTS; ++r) { acc[r][0] = acc[r][1] = acc[r][2] = acc[r][3] = 0.0; }
#pragma unroll 1
  for (int nl = 0; nl < cnt; ++nl) {
    const int n = g * a.gs + nl;
    const double e = s_eps[nl];
    const cplx* Xu = a.X + (ring + 2 * nl) * M + p0;
    const cplx* pu = a.psi + (size_t)(2 * n) * M + p0;
    cplx* ou = a.out + (size_t)(2 * n) * M + p0;
    if (MODE == F3_CORR) {
      const double sP = a.scale ? a.scale[n] : 1.0, ke = a.kappa * e, sn = s_sn[nl];
      const double cp = a.cpref[n], wa = a.w_a[n], wb = a.w_b[n];
#pragma unroll
      for (int r = 0; r < PTS; ++r) {
        const cplx xu = ldcg2(Xu + r * 128), xv = ldcg2(Xu + M + r * 128);
        const cplx wu = cscale(pu[r * 128], sP), wv = cscale(pu[M + r * 128], sP);
        const cplx u = make_double2((xu.x - ke * wu.y) * sn, (xu.y + ke * wu.x) * sn);
        const cplx v = make_double2((xv.x - ke * wv.y) * sn, (xv.y + ke * wv.x) * sn);
        ou[r * 128] = u; ou[M + r * 128] = v;
        if (a.do_dens) f3_dens_add(acc[r], u, v, cp, wa, wb);
      }
    } else {
#pragma unroll
      for (int r = 0; r < PTS; ++r) {
        const cplx yu = ldcg2(Xu + r * 128), yv = ldcg2(Xu + M + r * 128);
        const cplx u = pu[r * 128], v = pu[M + r * 128];
        ou[r * 128] = make_double2(yu.x - e * u.y, yu.y + e * u.x);
        ou[M + r * 128] = make_double2(yv.x - e * v.y, yv.y + e * v.x);
      }
    }
  }
  if (MODE == F3_CORR && a.do_dens) {
    double* ac = a.acc + (size_t)(g % F3_RING) * 4 * M + p0;
#pragma unroll
    for (int r = 0; r < PTS; ++r)
#pragma unroll
      for (int f = 0; f < 4; ++f) {
        double* q = ac + f * M + r * 128;
        *q = (g < F3_RING ? 0.0 : __ldcg(q)) + acc[r][f];
      }
  }
}

// ---- the persistent kernel ----------------------------------------------------------------------------------
template <bool SYM, int MODE>
__global__ void __launch_bounds__(128, 3) k_f3_mega(F3Mega a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* tiles = reinterpret_cast<cplx*>(smem_raw);
  __shared__ int s_item;
  __shared__ double red[4 * F3_NPART];
  __shared__ double s_eps[32], s_sn[32];
  cplx x[F3_N];
  const int G = a.G, NX = a.NX;
  int* done = reinterpret_cast<int*>(a.sync + 1);
  const int nA = a.gs * 2 * NX / 4, nB = a.gs * 16, nC = SYM ? a.gs * NX : a.gs * NX / 2;
  const int nD = MODE == F3_APPLY ? 0 : NX * F3_DSPLIT;
  const int IT = nA + nB + nC + nD, total = (G + 3) * IT;
  for (;;) {
    if (threadIdx.x == 0) s_item = atomicAdd(&a.sync->next, 1);
    __syncthreads();
    const int item = s_item;
    __syncthreads();
    if (item >= total) break;
    const int tick = item / IT, r = item - tick * IT;
    if (r < nA) {
      const int g = tick;
      if (g < G) {
        if (g >= F3_RING) f3_wait(&done[2 * G + g - F3_RING], nC, a.sync);
        f3_body_a<SYM>(a, g, r, tiles, x);
        f3_signal(&done[g]);
      }
    } else if (r < nA + nB) {
      const int g = tick - 1;
      if (g >= 0 && g < G) {
        f3_wait(&done[g], nA, a.sync);
        if (NX == 32) f3_body_b<32, SYM>(a, g, r - nA, x);
        else if (NX == 16) f3_body_b<16, SYM>(a, g, r - nA, x);
        else f3_body_b<8, SYM>(a, g, r - nA, x);
        f3_signal(&done[G + g]);
      }
    } else if (r < nA + nB + nC) {
      const int g = tick - 2;
      if (g >= 0 && g < G) {
        f3_wait(&done[G + g], nB, a.sync);
        if (MODE != F3_APPLY && g >= F3_RING) f3_wait(&done[3 * G + g - F3_RING], nD, a.sync);
        f3_body_c<SYM, MODE>(a, g, r - nA - nB, tiles, red, x);
        f3_signal(&done[2 * G + g]);
      }
    } else {
      const int g = tick - 3;
      if (g >= 0 && g < G) {
        f3_wait(&done[2 * G + g], nC, a.sync);
        if (g >= F3_RING) f3_wait(&done[3 * G + g - F3_RING], nD, a.sync);
        if (MODE != F3_APPLY) f3_body_d<MODE>(a, g, r - nA - nB - nC, s_eps, s_sn);
        f3_signal(&done[3 * G + g]);
      }
    }
  }
}
