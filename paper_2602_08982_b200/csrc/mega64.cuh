// mega64.cuh -- persistent dataflow stage kernels for the 64^3 lattice (configs[4]) with the Eq. 40 operator.
//
// Same scheme as mega3d.cuh (ticketed A/B/C/D work items, completion counters with release/acquire, spectrum rings
// with L2 eviction priorities), re-tiled for 64-point lines:
//  * a 64-point line is held by a PAIR of threads (lanes l and l ^ 16), 32 points each in registers: one radix-2
//    step across the pair through warp shuffles + the unrolled 32-point register transform of regfft.cuh.
//    Decimation in time takes an interleaved line (thread p holds points 2j + p) to a block spectrum (k + 32 p);
//    decimation in frequency takes block input to interleaved output, so forward (DIT) and inverse (DIF on the
//    conjugate) chain without any reordering.
//  * a 64 x 64 plane is 128 threads (4 warps) and one padded 64 x 65 tile; a CTA of 256 threads works on two
//    planes at a time (two x-planes in A, two kz rows in B, the two spectra  alpha lap w | lap(alpha w)  in C).
//  * the pipeline unit ("group") is ONE COMPONENT (4 MB, 8 MB of spectra), not a group of spinors: with five ring
//    slots about 45 MB are live, which the L2 can hold; D items run per spinor once both components are through C.
#pragma once
#include "mega3d.cuh"

#define F6_N 64
#define F6_PITCH 65
#define F6_PLANE (F6_N * F6_N)
#define F6_TILE (F6_N * F6_PITCH)
#define F6_RING 6
#define F6_THREADS 256
#define F6_M ((size_t)F6_N * F6_PLANE)
#define F6_ND 256              // D items per spinor (1024 points of both components each)

// d * exp(-2 pi i T / 64) for the odd member of the pair (p = 1), identity for the even one: branch-free
template <int T>
__device__ __forceinline__ cplx f6_tw(cplx d, int p) {
  const double c = p ? ws_cos64(T) : 1.0, s = p ? ws_sin64(T) : 0.0;
  return make_double2(fma(d.y, s, d.x * c), fma(-d.x, s, d.y * c));
}
__device__ __forceinline__ cplx f6_xchg(cplx v) {
  return make_double2(__shfl_xor_sync(0xffffffffu, v.x, 16), __shfl_xor_sync(0xffffffffu, v.y, 16));
}
template <int K>
struct F6Dit {                 // X[k] = E[k] + W^k O[k] (p = 0),  X[k + 32] = E[k] - W^k O[k] (p = 1)
  static __device__ __forceinline__ void run(cplx* x, int p) {
    const cplx t = f6_tw<K>(x[K], p), o = f6_xchg(t);
    x[K] = p ? csub(o, t) : cadd(t, o);
    if constexpr (K + 1 < 32) F6Dit<K + 1>::run(x, p);
  }
};
template <int J>
struct F6Dif {                 // even outputs from a + b (p = 0), odd outputs from (a - b) W^j (p = 1)
  static __device__ __forceinline__ void run(cplx* x, int p) {
    const cplx o = f6_xchg(x[J]);
    x[J] = p ? f6_tw<J>(csub(o, x[J]), 1) : cadd(x[J], o);
    if constexpr (J + 1 < 32) F6Dif<J + 1>::run(x, p);
  }
};
// interleaved line (x[j] = line[2 j + p]) -> block spectrum (x[k] = LINE[k + 32 p])
__device__ __forceinline__ void f6_dit(cplx* x, int p) { fft_reg<32, false>(x); F6Dit<0>::run(x, p); }
// block line (x[j] = line[j + 32 p]) -> interleaved spectrum (x[k] = LINE[2 k + p])
__device__ __forceinline__ void f6_dif(cplx* x, int p) { F6Dif<0>::run(x, p); fft_reg<32, false>(x); }

// barrier over the 128 threads of one half (h = 0, 1): the halves work on independent planes in the transforms,
// so they only meet at CTA-wide barriers where an item really needs both (C epilogue, dispatch)
__device__ __forceinline__ void f6_half_sync(int h) { asm volatile("bar.sync %0, 128;" :: "r"(h + 1) : "memory"); }

// forward 2-D transform of a plane held as interleaved lines along the slow axis (x[j] = (2 j + p, q)):
// returns x[k] = (k_fast = k + 32 p, k_slow = q).  S = the 128-thread group's tile; barriers over that group.  The two
// line transforms share one loop body so that the unrolled butterflies exist once per kernel site (instruction cache).
__device__ __forceinline__ void f6_plane_fwd(cplx* x, cplx* S, int q, int p, int h) {
#pragma unroll 1
  for (int pass = 0; pass < 2; ++pass) {
    f6_dit(x, p);
    if (pass == 0) {
#pragma unroll
      for (int k = 0; k < 32; ++k) S[(k + 32 * p) * F6_PITCH + q] = x[k];
      f6_half_sync(h);
#pragma unroll
      for (int j = 0; j < 32; ++j) x[j] = S[q * F6_PITCH + 2 * j + p];
      f6_half_sync(h);
    }
  }
}
// inverse counterpart on conjugated data: in x[j] = conj spectrum (k_fast = j + 32 p, k_slow = q), out x[k] = conj of
// the value at (slow = 2 k + p, fast = q)
__device__ __forceinline__ void f6_plane_inv(cplx* x, cplx* S, int q, int p, int h) {
#pragma unroll 1
  for (int pass = 0; pass < 2; ++pass) {
    f6_dif(x, p);
    if (pass == 0) {
#pragma unroll
      for (int k = 0; k < 32; ++k) S[(2 * k + p) * F6_PITCH + q] = x[k];
      f6_half_sync(h);
#pragma unroll
      for (int j = 0; j < 32; ++j) x[j] = S[q * F6_PITCH + j + 32 * p];
      f6_half_sync(h);
    }
  }
}

struct F6Mega {
  const cplx* psi;             // [n][2][M]
  const double* scale;         // per spinor (nullable)
  const double* kperp2;
  F3Fields F;
  const cplx* pack;            // [3][M] (k_f3_pack)
  const double *kx2, *ky2, *kz2;   // k_d^2, natural order (device tables)
  double invM, dV, kappa;
  cplx *spec0, *spec1, *X;     // rings [F6_RING][M]
  cplx* out;                   // APPLY: H psi; CORR: phi_new (= psi buffer); RHS: f_new
  const cplx* cpart;
  double* part;                // [F3_NPART][2 n * 64]   per (component group, x-plane)
  double* eps_out;
  int use_shift, normalize, do_dens;
  const double *cpref, *w_a, *w_b;
  double* acc;                 // ring [F6_RING][4][M]  (slot n % F6_RING)
  F3Sync* sync;                // followed by done[4][G]
  int n, G;                    // spinors, groups = 2 n
};

// thread coordinates inside the 128-thread half that owns a plane: line q in [0, 64), pair member p
struct F6Tid { int h, q, p; };
__device__ __forceinline__ F6Tid f6_tid() {
  const int tl = threadIdx.x & 127, lane = tl & 31;
  F6Tid t; t.h = threadIdx.x >> 7; t.p = lane >> 4; t.q = (tl >> 5) * 16 + (lane & 15);
  return t;
}

// ---- A: forward transforms of two x-planes of component group g (spectra of w and of alpha w) -------------------
__device__ __forceinline__ void f6_body_a(const F6Mega& a, const F3Pol& pol, int g, int ia, cplx* tiles, cplx* x) {
  const F6Tid t = f6_tid();
  const int n = g >> 1, c = g & 1, ix = 2 * ia + t.h;
  cplx* S = tiles + t.h * F6_TILE;
  const cplx* src = a.psi + ((size_t)g * F6_N + ix) * F6_PLANE;
  const double s = a.scale ? a.scale[n] : 1.0;
  const double* al = a.F.alpha[c] + (size_t)ix * F6_PLANE;
  const size_t sb = (size_t)(g % F6_RING) * F6_M + (size_t)ix * F6_PLANE;
#pragma unroll 1
  for (int tt = 0; tt < 2; ++tt) {
#pragma unroll
    for (int j = 0; j < 32; ++j) x[j] = ld_pol(src + (2 * j + t.p) * F6_N + t.q, pol.keep);
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      double f = s;
      if (tt) f *= al[(2 * j + t.p) * F6_N + t.q];
      x[j] = cscale(x[j], f);
    }
    f6_plane_fwd(x, S, t.q, t.p, t.h);
    cplx* dst = (tt == 0 ? a.spec0 : a.spec1) + sb;
#pragma unroll
    for (int k = 0; k < 32; ++k) st_pol(dst + (k + 32 * t.p) * F6_N + t.q, x[k], pol.keep);     // [kz][ky]
  }
}

// ---- B: x-lines of two kz rows: forward x, -k^2 / M, inverse x, in place (registers and shuffles only) ----------
__device__ __forceinline__ void f6_body_b(const F6Mega& a, const F3Pol& pol, int g, int ib, cplx* x) {
  const F6Tid t = f6_tid();
  const int kz = 2 * ib + t.h;
  const double kyz2 = a.ky2[t.q] + a.kz2[kz];
  const size_t sb = (size_t)(g % F6_RING) * F6_M + (size_t)kz * F6_N + t.q;
#pragma unroll 1
  for (int tt = 0; tt < 2; ++tt) {
    cplx* pz = (tt ? a.spec1 : a.spec0) + sb;
#pragma unroll
    for (int j = 0; j < 32; ++j) x[j] = ld_pol(pz + (size_t)(2 * j + t.p) * F6_PLANE, pol.keep);   // interleaved in x
    f6_dit(x, t.p);                                              // k_x = k + 32 p
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const double f = -(a.kx2[k + 32 * t.p] + kyz2) * a.invM;   // even derivative: Nyquist kept
      x[k] = make_double2(x[k].x * f, -x[k].y * f);              // conj for the inverse
    }
    f6_dif(x, t.p);                                              // conj of the values at x = 2 k + p
#pragma unroll
    for (int k = 0; k < 32; ++k) st_pol(pz + (size_t)(2 * k + t.p) * F6_PLANE, cconj(x[k]), pol.keep);
  }
}

// ---- C: one (component group, x-plane): the two halves invert  alpha lap w  and  lap(alpha w), then all 256 threads
// finish the BdG mix of that component (Eqs. 5, 15, 40) and the stage combination, 16 points each -----------------
template <int MODE>
__device__ __forceinline__ void f6_body_c(const F6Mega& a, const F3Pol& pol, int g, int ix, cplx* tiles, double* red, cplx* x) {
  const F6Tid t = f6_tid();
  const int n = g >> 1, c = g & 1, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const size_t pl = (size_t)ix * F6_PLANE, ring = (size_t)(g % F6_RING) * F6_M;
  cplx* S = tiles + t.h * F6_TILE;
  {
    const cplx* sp = (t.h ? a.spec1 : a.spec0) + ring + pl;
#pragma unroll
    for (int j = 0; j < 32; ++j) x[j] = ld_pol(sp + (j + 32 * t.p) * F6_N + t.q, pol.drop);   // (kz = j + 32 p, ky = q)
#pragma unroll
    for (int j = 0; j < 32; ++j) x[j] = cconj(x[j]);
    f6_plane_inv(x, S, t.q, t.p, t.h);                                  // conj of the value at (y = 2 k + p, z = q)
    const double* al = a.F.alpha[c] + pl;
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const int y = 2 * k + t.p;
      const double f = t.h == 0 ? al[y * F6_N + t.q] : 1.0;
      S[y * F6_PITCH + t.q] = make_double2(x[k].x * f, -x[k].y * f);
    }
  }
  __syncthreads();
  double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
  {
    const double s = a.scale ? a.scale[n] : 1.0, kp2 = a.kperp2[n];
    const cplx* pu = a.psi + (size_t)(2 * n) * F6_M + pl;
    const cplx* pv = pu + F6_M;
    cplx* oc = (MODE == F3_APPLY ? a.out + (size_t)g * F6_M : a.X + ring) + pl;
    const cplx* cc = a.cpart + (size_t)g * F6_M + pl;
    const cplx* pk = a.pack + pl;
#pragma unroll
    for (int r0 = 0; r0 < 16; r0 += 4) {
      cplx gu[4], gv[4], gq[4], gD[4], gA[4], g0[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int pt = (r0 + r) * F6_THREADS + tid;
        gu[r] = pu[pt]; gv[r] = pv[pt]; gq[r] = pk[pt]; gD[r] = pk[F6_M + pt];
        if (kp2 != 0.0) gA[r] = pk[2 * F6_M + pt];
        if (MODE == F3_CORR) g0[r] = cc[pt];
      }
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int pt = (r0 + r) * F6_THREADS + tid, si = (pt >> 6) * F6_PITCH + (pt & 63);
        const cplx u = cscale(gu[r], s), v = cscale(gv[r], s), w = c ? v : u;
        const cplx T0 = tiles[si], L1 = tiles[F6_TILE + si];
        double h = 0.5 * kp2;
        if (kp2 != 0.0) h *= c ? gA[r].y : gA[r].x;
        const cplx K = make_double2(-0.25 * (L1.x + T0.x) + h * w.x, -0.25 * (L1.y + T0.y) + h * w.y);   // Eq. 40 (lap alpha term in q)
        const cplx D = gD[r];
        cplx H;
        if (c == 0) H = cadd(K, cadd(cscale(u, gq[r].x), cmul(D, v)));                                    // Eqs. 5, 15
        else H = csub(cmul(cconj(D), u), cadd(K, cscale(v, gq[r].y)));
        e += w.x * H.x + w.y * H.y;
        if (MODE == F3_APPLY) st_pol_nb(oc + pt, H, pol.drop);
        else if (MODE == F3_RHS) st_pol_nb(oc + pt, make_double2(H.y, -H.x), pol.keep);
        else {
          const cplx X = make_double2(g0[r].x + a.kappa * H.y, g0[r].y - a.kappa * H.x);                  // C_part - i kappa H
          st_pol_nb(oc + pt, X, pol.keep);
          xx += cabs2(X); xpr += X.x * w.x + X.y * w.y; xpi += X.x * w.y - X.y * w.x; pp += cabs2(w);
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
  if (tid == 0) {
    const size_t np = (size_t)a.G * F6_N;
    for (int k = 0; k < (MODE == F3_CORR ? F3_NPART : 1); ++k) {
      double sum = 0.0;
      for (int w = 0; w < F6_THREADS / 32; ++w) sum += red[w * F3_NPART + k];
      a.part[k * np + (size_t)g * F6_N + ix] = sum;
    }
  }
}

// ---- D: per spinor n (dispatched with its odd component group): scalars from both components' partial sums, then
// 1024 points of both components per item: CORR phi_new = (X + i kappa eps w) s_n (+ densities), RHS f = Y + i eps phi --
template <int MODE, int NT = F6_THREADS>
__device__ __forceinline__ void f6_body_d(const F6Mega& a, const F3Pol& pol, int n, int id, double* s_sc) {
  const int tid = threadIdx.x, lane = tid & 31;
  const size_t np = (size_t)a.G * F6_N;
  if (tid < 32) {                                                  // warp 0: 2 x 64 partials per kind, fixed order
    double v[F3_NPART];
#pragma unroll
    for (int k = 0; k < F3_NPART; ++k) {
      double t = 0.0;
      if (k == 0 || MODE == F3_CORR) {
        const double* pp = a.part + k * np + (size_t)(2 * n) * F6_N;
        t = (__ldcg(pp + lane) + __ldcg(pp + 32 + lane)) + (__ldcg(pp + 64 + lane) + __ldcg(pp + 96 + lane));
      }
      v[k] = warp_sum(t);
    }
    if (lane == 0) {
      const double e_true = a.dV * v[0], e = a.use_shift ? e_true : 0.0;
      s_sc[0] = e; s_sc[1] = 1.0;
      if (id == 0 && a.eps_out) a.eps_out[n] = e_true;
      if (MODE == F3_CORR) {
        const double ke = a.kappa * e, nrm2 = a.dV * (v[1] - 2.0 * ke * v[3] + ke * ke * v[4]);
        s_sc[1] = a.normalize ? 1.0 / sqrt(nrm2) : 1.0;
      }
    }
  }
  __syncthreads();
  const double e = s_sc[0], sn = s_sc[1];
  const size_t p0 = (size_t)id * (4 * NT) + tid;
  const cplx* Xu = a.X + (size_t)((2 * n) % F6_RING) * F6_M + p0;
  const cplx* Xv = a.X + (size_t)((2 * n + 1) % F6_RING) * F6_M + p0;
  const cplx* pu = a.psi + (size_t)(2 * n) * F6_M + p0;
  cplx* ou = a.out + (size_t)(2 * n) * F6_M + p0;
  cplx gxu[4], gxv[4], gpu[4], gpv[4];
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    gxu[r] = __ldcg(Xu + r * NT); gxv[r] = __ldcg(Xv + r * NT); gpu[r] = pu[r * NT]; gpv[r] = pu[F6_M + r * NT];
  }
  if (MODE == F3_CORR) {
    const double sP = a.scale ? a.scale[n] : 1.0, ke = a.kappa * e;
    const double cp = a.cpref[n], wa = a.w_a[n], wb = a.w_b[n];
    double* ac = a.acc + (size_t)(n % F6_RING) * 4 * F6_M + p0;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const cplx wu = cscale(gpu[r], sP), wv = cscale(gpv[r], sP);
      const cplx u = make_double2((gxu[r].x - ke * wu.y) * sn, (gxu[r].y + ke * wu.x) * sn);
      const cplx v = make_double2((gxv[r].x - ke * wv.y) * sn, (gxv[r].y + ke * wv.x) * sn);
      st_pol_nb(ou + r * NT, u, pol.drop); st_pol_nb(ou + F6_M + r * NT, v, pol.drop);
      if (a.do_dens) {
        double d4[4] = {0.0, 0.0, 0.0, 0.0};
        f3_dens_add(d4, u, v, cp, wa, wb);
#pragma unroll
        for (int f = 0; f < 4; ++f) {
          double* qd = ac + f * F6_M + r * NT;
          *qd = (n < F6_RING ? 0.0 : __ldcg(qd)) + d4[f];
        }
      }
    }
  } else {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      st_pol_nb(ou + r * NT, make_double2(gxu[r].x - e * gpu[r].y, gxu[r].y + e * gpu[r].x), pol.drop);
      st_pol_nb(ou + F6_M + r * NT, make_double2(gxv[r].x - e * gpv[r].y, gxv[r].y + e * gpv[r].x), pol.drop);
    }
  }
}

// ---- the persistent kernel ----------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(F6_THREADS, 1) k_f6_mega(F6Mega a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* tiles = reinterpret_cast<cplx*>(smem_raw);
  __shared__ int s_item;
  __shared__ double red[(F6_THREADS / 32) * F3_NPART];
  __shared__ double s_sc[2];
  cplx x[32];
  const F3Pol pol = f3_policies();
  const int G = a.G;
  int* done = reinterpret_cast<int*>(a.sync + 1);
  const int nA = F6_N / 2, nB = F6_N / 2, nC = F6_N, nD = MODE == F3_APPLY ? 0 : F6_ND;
  const int IT = nA + nB + nC + nD, total = (G + 4) * IT;
  int t1 = 0;
  if (threadIdx.x == 0) t1 = atomicAdd(&a.sync->next, 1);
  for (;;) {
    if (threadIdx.x == 0) s_item = t1;
    __syncthreads();
    const int item = s_item;
    __syncthreads();
    if (item >= total) break;
    const int tick = item / IT, r = item - tick * IT;
    bool drew = false;
    if (r < nA) {
      const int g = tick;
      if (g < G) {
        if (g >= F6_RING) f3_wait(&done[2 * G + g - F6_RING], nC, a.sync);
        f6_body_a(a, pol, g, r, tiles, x);
        f3_signal(&done[g], &a.sync->next, t1); drew = true;
      }
    } else if (r < nA + nB) {
      const int g = tick - 1;
      if (g >= 0 && g < G) {
        f3_wait(&done[g], nA, a.sync);
        f6_body_b(a, pol, g, r - nA, x);
        f3_signal(&done[G + g], &a.sync->next, t1); drew = true;
      }
    } else if (r < nA + nB + nC) {
      const int g = tick - 2;
      if (g >= 0 && g < G) {
        f3_wait(&done[G + g], nB, a.sync);
        if (MODE != F3_APPLY && g >= F6_RING) f3_wait(&done[3 * G + ((g - F6_RING) | 1)], nD, a.sync);
        f6_body_c<MODE>(a, pol, g, r - nA - nB, tiles, red, x);
        f3_signal(&done[2 * G + g], &a.sync->next, t1); drew = true;
      }
    } else {
      const int g = tick - 4;
      if (g >= 0 && g < G && (g & 1)) {
        f3_wait(&done[2 * G + g], nC, a.sync);
        f3_wait(&done[2 * G + g - 1], nC, a.sync);
        if (a.do_dens && g >= 2 * F6_RING) f3_wait(&done[3 * G + g - 2 * F6_RING], nD, a.sync);
        if (MODE != F3_APPLY) f6_body_d<MODE>(a, pol, g >> 1, r - nA - nB - nC, s_sc);
        f3_signal(&done[3 * G + g], &a.sync->next, t1); drew = true;
      }
    }
    if (!drew && threadIdx.x == 0) t1 = atomicAdd(&a.sync->next, 1);
  }
}
