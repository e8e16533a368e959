// mega64s.cuh -- second tiling of the 64^3 persistent stage kernel: ONE plane per CTA (128 threads, one 64 x 65 tile,
// two independent CTAs per SM) instead of two planes in lock step per 256-thread CTA.
// The Eq. 40 C item is split so that every item needs a single tile and no CTA-wide hand-over between planes:
//   C0  inverse transform of the spectrum of w, times alpha           -> partial  alpha lap w  into the X ring slot
//   C1  inverse transform of the spectrum of alpha w; each thread then finishes ITS OWN 32 points straight from
//       registers (the values it holds after the transform): BdG mix, eps_n integrand, stage combination -> X ring / H psi
// Pipeline: A(t), B(t-1), C0(t-2), C1(t-3), D(spinor of the odd group t-5); groups are single components as in
// mega64.cuh; six ring slots.
#pragma once
#include "mega64.cuh"

#define F6S_THREADS 128
#define F6S_ND (F6_M / (4 * F6S_THREADS))     // D items per spinor: 512 points of both components each

struct F6STid { int q, p; };
__device__ __forceinline__ F6STid f6s_tid() {
  const int lane = threadIdx.x & 31;
  F6STid t; t.p = lane >> 4; t.q = (threadIdx.x >> 5) * 16 + (lane & 15);
  return t;
}
__device__ __forceinline__ void f6s_plane_fwd(cplx* x, cplx* S, int q, int p) {
#pragma unroll 1
  for (int pass = 0; pass < 2; ++pass) {
    f6_dit(x, p);
    if (pass == 0) {
#pragma unroll
      for (int k = 0; k < 32; ++k) S[(k + 32 * p) * F6_PITCH + q] = x[k];
      __syncthreads();
#pragma unroll
      for (int j = 0; j < 32; ++j) x[j] = S[q * F6_PITCH + 2 * j + p];
      __syncthreads();
    }
  }
}
__device__ __forceinline__ void f6s_plane_inv(cplx* x, cplx* S, int q, int p) {
#pragma unroll 1
  for (int pass = 0; pass < 2; ++pass) {
    f6_dif(x, p);
    if (pass == 0) {
#pragma unroll
      for (int k = 0; k < 32; ++k) S[(2 * k + p) * F6_PITCH + q] = x[k];
      __syncthreads();
#pragma unroll
      for (int j = 0; j < 32; ++j) x[j] = S[q * F6_PITCH + j + 32 * p];
      __syncthreads();
    }
  }
}

// ---- A: forward transforms (w and alpha w) of x-plane ix of component group g -----------------------------------
__device__ __forceinline__ void f6s_body_a(const F6Mega& a, const F3Pol& pol, int g, int ix, cplx* S, cplx* x) {
  const F6STid t = f6s_tid();
  const int n = g >> 1, c = g & 1;
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
    f6s_plane_fwd(x, S, t.q, t.p);
    cplx* dst = (tt == 0 ? a.spec0 : a.spec1) + sb;
#pragma unroll
    for (int k = 0; k < 32; ++k) st_pol(dst + (k + 32 * t.p) * F6_N + t.q, x[k], pol.keep);
  }
}

// ---- B: x-lines of the kz row of both spectra, in place ----------------------------------------------------------
__device__ __forceinline__ void f6s_body_b(const F6Mega& a, const F3Pol& pol, int g, int kz, cplx* x) {
  const F6STid t = f6s_tid();
  const double kyz2 = a.ky2[t.q] + a.kz2[kz];
  const size_t sb = (size_t)(g % F6_RING) * F6_M + (size_t)kz * F6_N + t.q;
#pragma unroll 1
  for (int tt = 0; tt < 2; ++tt) {
    cplx* pz = (tt ? a.spec1 : a.spec0) + sb;
#pragma unroll
    for (int j = 0; j < 32; ++j) x[j] = ld_pol(pz + (size_t)(2 * j + t.p) * F6_PLANE, pol.keep);
    f6_dit(x, t.p);
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const double f = -(a.kx2[k + 32 * t.p] + kyz2) * a.invM;
      x[k] = make_double2(x[k].x * f, -x[k].y * f);
    }
    f6_dif(x, t.p);
#pragma unroll
    for (int k = 0; k < 32; ++k) st_pol(pz + (size_t)(2 * k + t.p) * F6_PLANE, cconj(x[k]), pol.keep);
  }
}

// ---- C0: alpha lap w of plane ix -> partial in the X ring slot ---------------------------------------------------
__device__ __forceinline__ void f6s_body_c0(const F6Mega& a, const F3Pol& pol, int g, int ix, cplx* S, cplx* x) {
  const F6STid t = f6s_tid();
  const int c = g & 1;
  const size_t pl = (size_t)ix * F6_PLANE, ring = (size_t)(g % F6_RING) * F6_M;
  const cplx* sp = a.spec0 + ring + pl;
#pragma unroll
  for (int j = 0; j < 32; ++j) x[j] = ld_pol(sp + (j + 32 * t.p) * F6_N + t.q, pol.drop);
#pragma unroll
  for (int j = 0; j < 32; ++j) x[j] = cconj(x[j]);
  f6s_plane_inv(x, S, t.q, t.p);                                  // conj of lap w at (y = 2 k + p, z = q)
  const double* al = a.F.alpha[c] + pl;
  cplx* dst = a.X + ring + pl;
#pragma unroll
  for (int k = 0; k < 32; ++k) {
    const int i = (2 * k + t.p) * F6_N + t.q;
    const double f = al[i];
    st_pol(dst + i, make_double2(x[k].x * f, -x[k].y * f), pol.keep);
  }
}

// ---- C1: lap(alpha w) of plane ix, then each thread finishes its own 32 points (y = 2 k + p, z = q) ----------------
template <int MODE>
__device__ __forceinline__ void f6s_body_c1(const F6Mega& a, const F3Pol& pol, int g, int ix, cplx* S, double* red, cplx* x) {
  const F6STid t = f6s_tid();
  const int n = g >> 1, c = g & 1, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const size_t pl = (size_t)ix * F6_PLANE, ring = (size_t)(g % F6_RING) * F6_M;
  const cplx* sp = a.spec1 + ring + pl;
#pragma unroll
  for (int j = 0; j < 32; ++j) x[j] = ld_pol(sp + (j + 32 * t.p) * F6_N + t.q, pol.drop);
#pragma unroll
  for (int j = 0; j < 32; ++j) x[j] = cconj(x[j]);
  f6s_plane_inv(x, S, t.q, t.p);                                  // x[k] = conj of lap(alpha w) at (y = 2 k + p, z = q)
  double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
  const double s = a.scale ? a.scale[n] : 1.0, kp2 = a.kperp2[n];
  const cplx* pu = a.psi + (size_t)(2 * n) * F6_M + pl;
  const cplx* pv = pu + F6_M;
  cplx* part0 = a.X + ring + pl;                                   // alpha lap w from C0; overwritten by X / Y in place
  cplx* oc = (MODE == F3_APPLY ? a.out + (size_t)g * F6_M : a.X + ring) + pl;
  const cplx* cc = a.cpart + (size_t)g * F6_M + pl;
  const cplx* pk = a.pack + pl;
#pragma unroll
  for (int k0 = 0; k0 < 32; k0 += 4) {
    cplx gu[4], gv[4], gq[4], gD[4], gA[4], g0[4], gT[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int i = (2 * (k0 + r) + t.p) * F6_N + t.q;
      gu[r] = pu[i]; gv[r] = pv[i]; gq[r] = pk[i]; gD[r] = pk[F6_M + i]; gT[r] = __ldcg(part0 + i);
      if (kp2 != 0.0) gA[r] = pk[2 * F6_M + i];
      if (MODE == F3_CORR) g0[r] = cc[i];
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int i = (2 * (k0 + r) + t.p) * F6_N + t.q;
      const cplx u = cscale(gu[r], s), v = cscale(gv[r], s), w = c ? v : u;
      const cplx L1 = cconj(x[k0 + r]), T0 = gT[r];
      double h = 0.5 * kp2;
      if (kp2 != 0.0) h *= c ? gA[r].y : gA[r].x;
      const cplx K = make_double2(-0.25 * (L1.x + T0.x) + h * w.x, -0.25 * (L1.y + T0.y) + h * w.y);   // Eq. 40
      const cplx D = gD[r];
      cplx H;
      if (c == 0) H = cadd(K, cadd(cscale(u, gq[r].x), cmul(D, v)));                                    // Eqs. 5, 15
      else H = csub(cmul(cconj(D), u), cadd(K, cscale(v, gq[r].y)));
      e += w.x * H.x + w.y * H.y;
      if (MODE == F3_APPLY) st_pol_nb(oc + i, H, pol.drop);
      else if (MODE == F3_RHS) st_pol_nb(oc + i, make_double2(H.y, -H.x), pol.keep);
      else {
        const cplx X = make_double2(g0[r].x + a.kappa * H.y, g0[r].y - a.kappa * H.x);
        st_pol_nb(oc + i, X, pol.keep);
        xx += cabs2(X); xpr += X.x * w.x + X.y * w.y; xpi += X.x * w.y - X.y * w.x; pp += cabs2(w);
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
      for (int w = 0; w < F6S_THREADS / 32; ++w) sum += red[w * F3_NPART + k];
      a.part[k * np + (size_t)g * F6_N + ix] = sum;
    }
  }
}

// ---- the persistent kernel: done[kind][G], kinds A, B, C0, C1, D -------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(F6S_THREADS, 2) k_f6s_mega(F6Mega a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* S = reinterpret_cast<cplx*>(smem_raw);
  __shared__ int s_item;
  __shared__ double red[(F6S_THREADS / 32) * F3_NPART];
  __shared__ double s_sc[2];
  cplx x[32];
  const F3Pol pol = f3_policies();
  const int G = a.G;
  int* done = reinterpret_cast<int*>(a.sync + 1);
  const int nA = F6_N, nB = F6_N, nC = F6_N, nD = MODE == F3_APPLY ? 0 : (int)F6S_ND;
  const int IT = nA + nB + 2 * nC + nD, total = (G + 5) * IT;
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
        if (g >= F6_RING) f3_wait(&done[3 * G + g - F6_RING], nC, a.sync);           // spectra slot: C1 of its last user
        f6s_body_a(a, pol, g, r, S, x);
        f3_signal(&done[g], &a.sync->next, t1); drew = true;
      }
    } else if (r < nA + nB) {
      const int g = tick - 1;
      if (g >= 0 && g < G) {
        f3_wait(&done[g], nA, a.sync);
        f6s_body_b(a, pol, g, r - nA, x);
        f3_signal(&done[G + g], &a.sync->next, t1); drew = true;
      }
    } else if (r < nA + nB + nC) {
      const int g = tick - 2;
      if (g >= 0 && g < G) {
        f3_wait(&done[G + g], nB, a.sync);
        if (g >= F6_RING) {                                                          // X slot: last readers of its previous user
          f3_wait(&done[3 * G + g - F6_RING], nC, a.sync);
          if (MODE != F3_APPLY) f3_wait(&done[4 * G + ((g - F6_RING) | 1)], nD, a.sync);
        }
        f6s_body_c0(a, pol, g, r - nA - nB, S, x);
        f3_signal(&done[2 * G + g], &a.sync->next, t1); drew = true;
      }
    } else if (r < nA + nB + 2 * nC) {
      const int g = tick - 3;
      if (g >= 0 && g < G) {
        f3_wait(&done[2 * G + g], nC, a.sync);
        f6s_body_c1<MODE>(a, pol, g, r - nA - nB - nC, S, red, x);
        f3_signal(&done[3 * G + g], &a.sync->next, t1); drew = true;
      }
    } else {
      const int g = tick - 5;
      if (g >= 0 && g < G && (g & 1)) {
        f3_wait(&done[3 * G + g], nC, a.sync);
        f3_wait(&done[3 * G + g - 1], nC, a.sync);
        if (a.do_dens && g >= 2 * F6_RING) f3_wait(&done[4 * G + g - 2 * F6_RING], nD, a.sync);
        if (MODE != F3_APPLY) f6_body_d<MODE, F6S_THREADS>(a, pol, g >> 1, r - nA - nB - 2 * nC, s_sc);
        f3_signal(&done[4 * G + g], &a.sync->next, t1); drew = true;
      }
    }
    if (!drew && threadIdx.x == 0) t1 = atomicAdd(&a.sync->next, 1);
  }
}
