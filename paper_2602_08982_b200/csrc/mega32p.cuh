// mega32p.cuh -- the 32^3 persistent stage kernel with PAIR-OF-THREADS lines (16 points per thread).
//
// Same dataflow as mega3d.cuh (ticketed A/B/C/D items over groups of gs spinors, ring of 4 slots) and the same
// result; what changes is the tiling: a 32-point line is held by two threads (lanes l and l ^ 16, one radix-2
// step through warp shuffles + the unrolled 16-point register transform), so a thread needs about 110 registers
// instead of 255 and an SM holds 16 warps instead of 8 for the same number of planes in flight -- the same L2
// footprint with twice the warps to hide the L2 / HBM latency that bounds mega3d (profiles/r01_ncu_mega_*.md).
// A 32 x 32 plane is 64 threads and one padded 32 x 33 tile; a CTA of 256 threads works on four planes at a time:
// four component planes in A, four (component, kz) rows in B, the four spectra of one (spinor, x-plane) in C.
#pragma once
#include "mega3d.cuh"

#define F5_THREADS 256

template <int K>
__device__ __forceinline__ cplx f5_tw(cplx d, int p) {          // d * exp(-2 pi i K / 32) for p = 1, identity for p = 0
  const double c = p ? ws_cos64(2 * K) : 1.0, s = p ? ws_sin64(2 * K) : 0.0;
  return make_double2(fma(d.y, s, d.x * c), fma(-d.x, s, d.y * c));
}
__device__ __forceinline__ cplx f5_xchg(cplx v) {
  return make_double2(__shfl_xor_sync(0xffffffffu, v.x, 16), __shfl_xor_sync(0xffffffffu, v.y, 16));
}
template <int K>
struct F5Dit {
  static __device__ __forceinline__ void run(cplx* x, int p) {
    const cplx t = f5_tw<K>(x[K], p), o = f5_xchg(t);
    x[K] = p ? csub(o, t) : cadd(t, o);
    if constexpr (K + 1 < 16) F5Dit<K + 1>::run(x, p);
  }
};
template <int J>
struct F5Dif {
  static __device__ __forceinline__ void run(cplx* x, int p) {
    const cplx o = f5_xchg(x[J]);
    x[J] = p ? f5_tw<J>(csub(o, x[J]), 1) : cadd(x[J], o);
    if constexpr (J + 1 < 16) F5Dif<J + 1>::run(x, p);
  }
};
// interleaved line (x[j] = line[2 j + p]) -> block spectrum (x[k] = LINE[k + 16 p])
__device__ __forceinline__ void f5_dit(cplx* x, int p) { fft_reg<16, false>(x); F5Dit<0>::run(x, p); }
// block line (x[j] = line[j + 16 p]) -> interleaved spectrum (x[k] = LINE[2 k + p])
__device__ __forceinline__ void f5_dif(cplx* x, int p) { F5Dif<0>::run(x, p); fft_reg<16, false>(x); }

// barrier over the 64 threads that own one plane (quarter h of the CTA)
__device__ __forceinline__ void f5_quarter_sync(int h) { asm volatile("bar.sync %0, 64;" :: "r"(h + 1) : "memory"); }

struct F5Tid { int h, q, p; };                                   // quarter, line in [0, 32), pair member
__device__ __forceinline__ F5Tid f5_tid() {
  const int tl = threadIdx.x & 63, lane = tl & 31;
  F5Tid t; t.h = threadIdx.x >> 6; t.p = lane >> 4; t.q = (tl >> 5) * 16 + (lane & 15);
  return t;
}

// forward plane transform: in x[j] = (slow = 2 j + p, fast = q), out x[k] = (k_fast = k + 16 p, k_slow = q)
__device__ __forceinline__ void f5_plane_fwd(cplx* x, cplx* S, const F5Tid& t) {
#pragma unroll 1
  for (int pass = 0; pass < 2; ++pass) {
    f5_dit(x, t.p);
    if (pass == 0) {
#pragma unroll
      for (int k = 0; k < 16; ++k) S[(k + 16 * t.p) * F3_PITCH + t.q] = x[k];
      f5_quarter_sync(t.h);
#pragma unroll
      for (int j = 0; j < 16; ++j) x[j] = S[t.q * F3_PITCH + 2 * j + t.p];
      f5_quarter_sync(t.h);
    }
  }
}
// inverse on conjugated data: in x[j] = conj spectrum (k_fast = j + 16 p, k_slow = q), out conj value (slow = 2 k + p, fast = q)
__device__ __forceinline__ void f5_plane_inv(cplx* x, cplx* S, const F5Tid& t) {
#pragma unroll 1
  for (int pass = 0; pass < 2; ++pass) {
    f5_dif(x, t.p);
    if (pass == 0) {
#pragma unroll
      for (int k = 0; k < 16; ++k) S[(2 * k + t.p) * F3_PITCH + t.q] = x[k];
      f5_quarter_sync(t.h);
#pragma unroll
      for (int j = 0; j < 16; ++j) x[j] = S[t.q * F3_PITCH + j + 16 * t.p];
      f5_quarter_sync(t.h);
    }
  }
}

// ---- A: forward transforms of four component planes (one per quarter) ------------------------------------------
template <bool SYM>
__device__ __forceinline__ void f5_body_a(const F3Mega& a, const F3Pol& pol, int g, int ia, cplx* tiles, cplx* x) {
  const F5Tid t = f5_tid();
  const int pi = 4 * ia + t.h, nl = pi >> 6, rem = pi & 63, c = rem >> 5, ix = rem & 31, n = g * a.gs + nl;
  if (n >= a.n) return;                                          // quarter-uniform; only quarter barriers follow
  cplx* S = tiles + t.h * (F3_N * F3_PITCH);
  const size_t M = (size_t)F3_N * F3_PLANE;
  const cplx* src = a.psi + ((size_t)(2 * n + c) * F3_N + ix) * F3_PLANE;
  const double s = a.scale ? a.scale[n] : 1.0;
  const double* al = a.F.alpha[c] + (size_t)ix * F3_PLANE;
  const size_t sb = (((size_t)(g % F3_RING) * a.gs + nl) * 2 + c) * M + (size_t)ix * F3_PLANE;
#pragma unroll 1
  for (int tt = 0; tt < (SYM ? 2 : 1); ++tt) {
#pragma unroll
    for (int j = 0; j < 16; ++j) x[j] = ld_pol(src + (2 * j + t.p) * F3_N + t.q, pol.keep);
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      double f = s;
      if (SYM && tt) f *= al[(2 * j + t.p) * F3_N + t.q];
      x[j] = cscale(x[j], f);
    }
    f5_plane_fwd(x, S, t);
    cplx* dst = (tt == 0 ? a.spec0 : a.spec1) + sb;
#pragma unroll
    for (int k = 0; k < 16; ++k) st_pol(dst + (k + 16 * t.p) * F3_N + t.q, x[k], pol.keep);      // [kz][ky]
  }
}

// ---- B: x-lines of four (component, kz) rows, in place -----------------------------------------------------------
template <bool SYM>
__device__ __forceinline__ void f5_body_b(const F3Mega& a, const F3Pol& pol, int g, int ib, cplx* x) {
  const F5Tid t = f5_tid();
  const int ri = 4 * ib + t.h, kz = ri & 31, ccl = ri >> 5;
  if (g * a.gs + (ccl >> 1) >= a.n) return;
  const size_t M = (size_t)F3_N * F3_PLANE;
  const double kyz2 = a.ky2[t.q] + a.kz2[kz];
  const size_t sb = ((size_t)(g % F3_RING) * a.gs * 2 + ccl) * M + kz * F3_N + t.q;
#pragma unroll 1
  for (int tt = 0; tt < (SYM ? 2 : 1); ++tt) {
    cplx* pz = (tt ? a.spec1 : a.spec0) + sb;
#pragma unroll
    for (int j = 0; j < 16; ++j) x[j] = ld_pol(pz + (size_t)(2 * j + t.p) * F3_PLANE, pol.keep);
    f5_dit(x, t.p);                                              // k_x = k + 16 p
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const double f = -((t.p ? a.kx2[k + 16] : a.kx2[k]) + kyz2) * a.invM;
      x[k] = make_double2(x[k].x * f, -x[k].y * f);
    }
    f5_dif(x, t.p);                                              // conj of the values at x = 2 k + p
#pragma unroll
    for (int k = 0; k < 16; ++k) st_pol(pz + (size_t)(2 * k + t.p) * F3_PLANE, cconj(x[k]), pol.keep);
  }
}

// ---- C: the quarters invert  alpha lap u | lap(alpha u) | alpha lap v | lap(alpha v)  of one (spinor, x-plane)
// (Eq. 14: lap u | lap v of two planes), leave them in their tiles, and after the CTA barrier every thread finishes
// 4 (8) points of both components: BdG mix, eps_n integrand, stage combination -----------------------------------
template <bool SYM, int MODE>
__device__ __forceinline__ void f5_body_c(const F3Mega& a, const F3Pol& pol, int g, int ic, cplx* tiles, double* red, cplx* x) {
  constexpr int NS = SYM ? 2 : 1, QPI = 2 * NS, IPC = 4 / QPI, TPI = 64 * QPI, PPT = F3_PLANE / TPI, TILE = F3_N * F3_PITCH;
  const F5Tid t = f5_tid();
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int pI = t.h / QPI, hl = t.h % QPI, c = hl / NS, tt = hl % NS;
  const int item = ic * IPC + pI, nl = item >> 5, ix = item & 31, n = g * a.gs + nl;
  const bool valid = n < a.n;
  const size_t M = (size_t)F3_N * F3_PLANE, pl = (size_t)ix * F3_PLANE;
  const size_t ring = ((size_t)(g % F3_RING) * a.gs + nl) * 2;
  cplx* S = tiles + t.h * TILE;
  if (valid) {
    const cplx* sp = (tt ? a.spec1 : a.spec0) + (ring + c) * M + pl;
#pragma unroll
    for (int j = 0; j < 16; ++j) x[j] = ld_pol(sp + (j + 16 * t.p) * F3_N + t.q, pol.drop);      // (kz = j + 16 p, ky = q)
#pragma unroll
    for (int j = 0; j < 16; ++j) x[j] = cconj(x[j]);
    f5_plane_inv(x, S, t);                                         // conj of the value at (y = 2 k + p, z = q)
    const double* al = a.F.alpha[c] + pl;
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int y = 2 * k + t.p;
      const double f = (SYM && tt == 0) ? al[y * F3_N + t.q] : 1.0;
      S[y * F3_PITCH + t.q] = make_double2(x[k].x * f, -x[k].y * f);
    }
  }
  __syncthreads();
  double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
  if (valid) {
    const int tl = tid - pI * TPI;                                 // thread index inside the item's group
    const cplx* tb = tiles + pI * QPI * TILE;
    const double s = a.scale ? a.scale[n] : 1.0, kp2 = a.kperp2[n];
    const cplx* pu = a.psi + (size_t)(2 * n) * M + pl;
    const cplx* pv = pu + M;
    cplx* ou = (MODE == F3_APPLY ? a.out + (size_t)(2 * n) * M : a.X + ring * M) + pl;
    cplx* ov = ou + M;
    const cplx* cu = a.cpart + (size_t)(2 * n) * M + pl;
    const cplx* pk = a.pack + pl;
#pragma unroll
    for (int r0 = 0; r0 < PPT; r0 += 4) {
      cplx gu[4], gv[4], gq[4], gD[4], gA[4], g0[4], g1[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int i = (r0 + r) * TPI + tl;
        gu[r] = pu[i]; gv[r] = pv[i]; gq[r] = pk[i]; gD[r] = pk[M + i];
        if (SYM && kp2 != 0.0) gA[r] = pk[2 * M + i];
        if (MODE == F3_CORR) { g0[r] = cu[i]; g1[r] = cu[M + i]; }
      }
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int i = (r0 + r) * TPI + tl, si = (i >> 5) * F3_PITCH + (i & 31);
        const cplx u = cscale(gu[r], s), v = cscale(gv[r], s);
        const cplx Lu = tb[(NS - 1) * TILE + si], Lv = tb[(2 * NS - 1) * TILE + si];
        const cplx q = gq[r], D = gD[r];
        double ha = 0.5 * kp2, hb = 0.5 * kp2;
        if (SYM && kp2 != 0.0) { ha *= gA[r].x; hb *= gA[r].y; }
        cplx Ku, Kv;
        if (SYM) {                                                 // Eq. 40; its +(lap alpha) w / 4 term sits in q
          const cplx Tu = tb[si], Tv = tb[NS * TILE + si];
          Ku = make_double2(-0.25 * (Lu.x + Tu.x) + ha * u.x, -0.25 * (Lu.y + Tu.y) + ha * u.y);
          Kv = make_double2(-0.25 * (Lv.x + Tv.x) + hb * v.x, -0.25 * (Lv.y + Tv.y) + hb * v.y);
        } else {                                                   // Eq. 14
          Ku = make_double2(-0.5 * Lu.x + ha * u.x, -0.5 * Lu.y + ha * u.y);
          Kv = make_double2(-0.5 * Lv.x + hb * v.x, -0.5 * Lv.y + hb * v.y);
        }
        const cplx Hu = cadd(Ku, cadd(cscale(u, q.x), cmul(D, v)));                             // Eqs. 5, 15
        const cplx Hv = csub(cmul(cconj(D), u), cadd(Kv, cscale(v, q.y)));
        e += u.x * Hu.x + u.y * Hu.y + v.x * Hv.x + v.y * Hv.y;
        if (MODE == F3_APPLY) { st_pol_nb(ou + i, Hu, pol.drop); st_pol_nb(ov + i, Hv, pol.drop); }
        else if (MODE == F3_RHS) { st_pol_nb(ou + i, make_double2(Hu.y, -Hu.x), pol.keep); st_pol_nb(ov + i, make_double2(Hv.y, -Hv.x), pol.keep); }
        else {
          const cplx xu = make_double2(g0[r].x + a.kappa * Hu.y, g0[r].y - a.kappa * Hu.x);     // C_part - i kappa H
          const cplx xv = make_double2(g1[r].x + a.kappa * Hv.y, g1[r].y - a.kappa * Hv.x);
          st_pol_nb(ou + i, xu, pol.keep); st_pol_nb(ov + i, xv, pol.keep);
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
    red[warp * F3_NPART] = e;
    if (MODE == F3_CORR) { red[warp * F3_NPART + 1] = xx; red[warp * F3_NPART + 2] = xpr; red[warp * F3_NPART + 3] = xpi; red[warp * F3_NPART + 4] = pp; }
  }
  __syncthreads();
  if (valid && tid == pI * TPI) {
    constexpr int WPI = TPI / 32;
    const size_t np = (size_t)a.n * F3_N;
    for (int k = 0; k < (MODE == F3_CORR ? F3_NPART : 1); ++k) {
      double sum = 0.0;
      for (int w = 0; w < WPI; ++w) sum += red[(pI * WPI + w) * F3_NPART + k];
      a.part[k * np + (size_t)n * F3_N + ix] = sum;
    }
  }
}

// ---- the persistent kernel ----------------------------------------------------------------------------------
template <bool SYM, int MODE>
__global__ void __launch_bounds__(F5_THREADS, 2) k_f5_mega(F3Mega a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* tiles = reinterpret_cast<cplx*>(smem_raw);
  __shared__ int s_item[2];
  __shared__ double red[(F5_THREADS / 32) * F3_NPART];
  __shared__ double s_eps[32], s_sn[32];
  cplx x[16];
  const F3Pol pol = f3_policies();
  const int G = a.G;
  int* done = reinterpret_cast<int*>(a.sync + 1);
  const int nA = a.gs * 16, nB = a.gs * 16, nC = SYM ? a.gs * F3_N : a.gs * F3_N / 2;
  const int nD = MODE == F3_APPLY ? 0 : F3_N * F3_DSPLIT;
  const int IT = nA + nB + nC + nD, total = (G + 3) * IT;
  const int pf_lines = a.gs * 2 * F3_N * (F3_PLANE * 16 / 128), pf_chunk = (pf_lines + IT - 1) / IT;
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
    f3_prefetch_tick<MODE, F5_THREADS>(a, tick, r, pf_chunk, pf_lines);
    if (r < nA) {
      const int g = tick;
      if (g < G) {
        if (g >= F3_RING) f3_wait(&done[2 * G + g - F3_RING], nC, a.sync);
        f5_body_a<SYM>(a, pol, g, r, tiles, x);
        f3_signal(&done[g], &a.sync->next, t1); drew = true;
      }
    } else if (r < nA + nB) {
      const int g = tick - 1;
      if (g >= 0 && g < G) {
        f3_wait(&done[g], nA, a.sync);
        f5_body_b<SYM>(a, pol, g, r - nA, x);
        f3_signal(&done[G + g], &a.sync->next, t1); drew = true;
      }
    } else if (r < nA + nB + nC) {
      const int g = tick - 2;
      if (g >= 0 && g < G) {
        f3_wait(&done[G + g], nB, a.sync);
        if (MODE != F3_APPLY && g >= F3_RING) f3_wait(&done[3 * G + g - F3_RING], nD, a.sync);
        f5_body_c<SYM, MODE>(a, pol, g, r - nA - nB, tiles, red, x);
        f3_signal(&done[2 * G + g], &a.sync->next, t1); drew = true;
      }
    } else {
      const int g = tick - 3;
      if (g >= 0 && g < G) {
        f3_wait(&done[2 * G + g], nC, a.sync);
        if (g >= F3_RING) f3_wait(&done[3 * G + g - F3_RING], nD, a.sync);
        if (MODE != F3_APPLY) f3_body_d<MODE, F5_THREADS>(a, pol, g, r - nA - nB - nC, s_eps, s_sn);
        f3_signal(&done[3 * G + g], &a.sync->next, t1); drew = true;
      }
    }
    if (!drew && threadIdx.x == 0) t1 = atomicAdd(&a.sync->next, 1);
  }
}
