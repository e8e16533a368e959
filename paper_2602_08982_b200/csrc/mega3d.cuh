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
// optional phase timing (build with -DF3_TIMING): per-kind cycle sums in g_f3_cycles[kind][phase]
#ifdef F3_TIMING
__device__ unsigned long long g_f3_cycles[8][8];
#define F3_T0() long long t_ = clock64()
#define F3_T(kind, phase) do { long long n_ = clock64(); if ((threadIdx.x & 31) == 0) atomicAdd(&g_f3_cycles[kind][phase], (unsigned long long)(n_ - t_)); t_ = n_; } while (0)
#else
#define F3_T0() do {} while (0)
#define F3_T(kind, phase) do {} while (0)
#endif
#define F3_MEGA_OCC 2
#ifndef F3_DSPLIT
#define F3_DSPLIT 2            // D items per x-plane
#endif

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
  const cplx* pack;            // [3][M]: (q_a, q_b), Delta + Delta_ext, (alpha_a, alpha_b)  -- see k_f3_pack
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

// Pointwise fields of H gathered per lattice point so that the C epilogue reads 2-3 16-byte words instead of
// ten scattered ones: q_sigma = U_sigma - mu_sigma (+ lap(alpha_sigma) / 4 for the Eq. 40 form, whose
// -(lap alpha) w / 4... term enters H with +1/4), D = Delta + Delta_ext, and alpha_sigma for the transverse shift.
__global__ void k_f3_pack(F3Fields F, int sym, int64_t M, cplx* pack) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  const double qa = F.U[0][i] - F.mu[0] + (sym ? 0.25 * F.lap[0][i] : 0.0);
  const double qb = F.U[1][i] - F.mu[1] + (sym ? 0.25 * F.lap[1][i] : 0.0);
  pack[i] = make_double2(qa, qb);
  pack[M + i] = cadd(F.delta[i], F.dext[i]);
  pack[2 * M + i] = make_double2(F.alpha[0][i], F.alpha[1][i]);
}

__device__ __forceinline__ cplx ldcg2(const cplx* p) { return __ldcg(p); }

// L2 eviction priorities (createpolicy, PTX ISA 7.4+): the spectrum / X rings and psi are re-read by later items
// and must survive in L2 (evict_last); data touched for the last time is marked evict_first so that it leaves
// first.  KEEP / DROP are per-thread 64-bit policy words.
struct F3Pol { uint64_t keep, drop; };
__device__ __forceinline__ F3Pol f3_policies() {
  F3Pol p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p.keep));
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p.drop));
  return p;
}
__device__ __forceinline__ cplx ld_pol(const cplx* p, uint64_t pol) {        // L1-bypassing load with an L2 policy
  cplx v;
  asm volatile("ld.global.cg.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ void st_pol(cplx* p, cplx v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" :: "l"(p), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}

// same store without the compiler memory barrier: lets the plain loads of the next loop iterations be hoisted above it
// (volatile asm statements keep their order among themselves, ordinary loads may pass them)
__device__ __forceinline__ void st_pol_nb(cplx* p, cplx v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1, %2}, %3;" :: "l"(p), "d"(v.x), "d"(v.y), "l"(pol));
}

__device__ __forceinline__ void f3_pf1(const void* p) { asm volatile("prefetch.global.L1 [%0];" :: "l"(p)); }
__device__ __forceinline__ void f3_pf(const void* p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }


// one thread waits until *ctr >= target (bounded), then the whole CTA proceeds.  The counter is read with acquire
// semantics (no separate fence) and bumped with a release reduction: the PTX memory model's release/acquire pair on
// the counter orders the producers' stores (made visible to thread 0 by the CTA barrier) before the consumers' loads.
// (Deferring the release into the next item's load phase was measured: it hides the release latency but delays the
// dependants more than it saves.)
__device__ __forceinline__ int f3_ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void f3_red_release(int* p) {
  asm volatile("red.release.gpu.global.add.s32 [%0], 1;" :: "l"(p) : "memory");
}
__constant__ int g_f3_spin_limit = 1 << 25;      // polls of 200 ns (about 7 s); wslda_tuning.spin_limit, set at context creation
__device__ __forceinline__ void f3_wait(int* ctr, int target, F3Sync* sy) {
  if (threadIdx.x == 0) {
    int spins = 0;
    while (f3_ld_acquire(ctr) < target) {
      __nanosleep(200);
      if (++spins > g_f3_spin_limit) { sy->error = 1; break; }    // the host reads the flag after the launch (ctx.cuh cuda_check)
    }
  }
  __syncthreads();
}
__device__ __forceinline__ void f3_signal(int* ctr, int* next, int& ticket) {
  if (threadIdx.x == 0) ticket = atomicAdd(next, 1);       // the next ticket travels while the barrier and the release complete
  __syncthreads();
  if (threadIdx.x == 0) f3_red_release(ctr);
}

// ---- A: forward plane transforms of 4 component planes (one per warp) ----------------------------------------
template <bool SYM>
__device__ __forceinline__ void f3_body_a(const F3Mega& a, const F3Pol& pol, int g, int ia, cplx* tiles, cplx* x) {
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
  F3_T0();
#pragma unroll 1
  for (int t = 0; t < (SYM ? 2 : 1); ++t) {
#pragma unroll
    for (int j = 0; j < F3_N; ++j) {
      double f = s;
      if (SYM && t) f *= al[j * F3_N + lane];
      x[j] = cscale(ld_pol(src + j * F3_N + lane, pol.keep), f);      // psi is read again by C (and D)
    }
    F3_T(0, 0);
    f3_plane_forward(x, S, lane);
    F3_T(0, 1);
    cplx* dst = (t == 0 ? a.spec0 : a.spec1) + sb;
#pragma unroll
    for (int j = 0; j < F3_N; ++j) st_pol(dst + j * F3_N + lane, x[j], pol.keep);
    F3_T(0, 2);
  }
}

// ---- B: x-lines of 4 (component, kz) rows: FFT x, -k^2/M, inverse FFT x, in place ------------------------------
template <int NX, bool SYM>
__device__ __forceinline__ void f3_body_b(const F3Mega& a, const F3Pol& pol, int g, int ib, cplx* x) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q = 4 * ib + warp, kz = q & (F3_N - 1), ccl = q >> 5;
  if (g * a.gs + (ccl >> 1) >= a.n) return;
  const size_t M = (size_t)NX * F3_PLANE;
  const double kyz2 = a.ky2[lane] + a.kz2[kz];
  const size_t sb = ((size_t)(g % F3_RING) * a.gs * 2 + ccl) * M + kz * F3_N + lane;
  F3_T0();
#pragma unroll 1
  for (int t = 0; t < (SYM ? 2 : 1); ++t) {
    cplx* p = (t ? a.spec1 : a.spec0) + sb;
#pragma unroll
    for (int j = 0; j < NX; ++j) x[j] = ld_pol(p + (size_t)j * F3_PLANE, pol.keep);
    F3_T(1, 0);
#pragma unroll 1
    for (int dir = 0; dir < 2; ++dir) {
      fft_reg<NX, false>(x);
#pragma unroll
      for (int j = 0; j < NX; ++j) {
        const double f = dir ? 1.0 : -(a.kx2[j] + kyz2) * a.invM;
        x[j] = make_double2(x[j].x * f, -x[j].y * f);
      }
    }
    F3_T(1, 1);
#pragma unroll
    for (int j = 0; j < NX; ++j) st_pol(p + (size_t)j * F3_PLANE, x[j], pol.keep);
    F3_T(1, 2);
  }
}

// ---- C: inverse plane transforms (one per warp), then the pointwise BdG mix and the stage combination ----------
// SYM: the 4 warps hold alpha lap u | lap(alpha u) | alpha lap v | lap(alpha v) of ONE (spinor, x-plane);
// Eq. 14: lap u | lap v of TWO x-planes.  Each warp leaves its plane in its own tile; after the barrier every
// thread finishes 32 / WPI rows of both components (psi, C_part and the fields are read once per point).
template <bool SYM, int MODE>
__device__ __forceinline__ void f3_body_c(const F3Mega& a, const F3Pol& pol, int g, int ic, cplx* tiles, double* red, cplx* x) {
  constexpr int NS = SYM ? 2 : 1, WPI = 2 * NS, IPC = 4 / WPI, ROWS = F3_N / WPI, TILE = F3_N * F3_PITCH;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int pI = warp / WPI, wl = warp % WPI, c = wl / NS, t = wl % NS;
  const int item = ic * IPC + pI, nl = item / a.NX, ix = item - nl * a.NX, n = g * a.gs + nl;
  const bool valid = n < a.n;
  const size_t M = (size_t)a.NX * F3_PLANE, pl = (size_t)ix * F3_PLANE;
  const size_t ring = ((size_t)(g % F3_RING) * a.gs + nl) * 2;        // ring index of component 0 of this spinor
  cplx* S = tiles + warp * TILE;
  F3_T0();
  if (valid) {
    // this thread's epilogue rows: pull psi, C_part and the fields towards L1 now, they are used after the transform
    {
      const size_t r0 = pl + (size_t)(wl * ROWS) * F3_N;             // first point of the warp's rows
      const char* pu8 = (const char*)(a.psi + (size_t)(2 * n) * M + r0);
      const char* cu8 = (const char*)(a.cpart + (size_t)(2 * n) * M + r0);
      constexpr int LW = ROWS * F3_N * 16 / 128;                     // 128-byte lines of complex rows per warp
      for (int q = lane; q < LW; q += 32) {
        f3_pf1(pu8 + q * 128); f3_pf1(pu8 + M * 16 + q * 128);
        if (MODE == F3_CORR) { f3_pf1(cu8 + q * 128); f3_pf1(cu8 + M * 16 + q * 128); }
      }
      for (int q = lane; q < LW; q += 32) { f3_pf1((const char*)(a.pack + r0) + q * 128); f3_pf1((const char*)(a.pack + M + r0) + q * 128); }
    }
    const cplx* sp = (t ? a.spec1 : a.spec0) + (ring + c) * M + pl;
#pragma unroll
    for (int j = 0; j < F3_N; ++j) x[j] = cconj(ld_pol(sp + j * F3_N + lane, pol.drop));        // last use of the spectrum
    F3_T(2, 0);
    f3_plane_forward(x, S, lane);                                    // conj of the value at (y = j, z = lane)
    F3_T(2, 1);
    const double* al = a.F.alpha[c] + pl;
#pragma unroll
    for (int j = 0; j < F3_N; ++j) {
      const double f = (SYM && t == 0) ? al[j * F3_N + lane] : 1.0;
      S[j * F3_PITCH + lane] = make_double2(x[j].x * f, -x[j].y * f);
    }
  }
  F3_T(2, 2);
  __syncthreads();
  F3_T(2, 3);
  double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
  if (valid) {
    const cplx* tb = tiles + pI * WPI * TILE;
    const double s = a.scale ? a.scale[n] : 1.0, kp2 = a.kperp2[n];
    const cplx* pu = a.psi + (size_t)(2 * n) * M + pl;
    const cplx* pv = pu + M;
    cplx* ou = (MODE == F3_APPLY ? a.out + (size_t)(2 * n) * M : a.X + ring * M) + pl;
    cplx* ov = ou + M;
    const cplx* cu = a.cpart + (size_t)(2 * n) * M + pl;
    const cplx* pk = a.pack + pl;
#pragma unroll
    for (int jj0 = 0; jj0 < ROWS; jj0 += 4) {
     // four rows at a time: every global load of the chunk is issued before the first use
     cplx gu[4], gv[4], gq[4], gD[4], gA[4], g0[4], g1[4];
#pragma unroll
     for (int r = 0; r < 4; ++r) {
       const int i = (wl * ROWS + jj0 + r) * F3_N + lane;
       gu[r] = pu[i]; gv[r] = pv[i]; gq[r] = pk[i]; gD[r] = pk[M + i];
       if (SYM && kp2 != 0.0) gA[r] = pk[2 * M + i];
       if (MODE == F3_CORR) { g0[r] = cu[i]; g1[r] = cu[M + i]; }
     }
#pragma unroll
     for (int r = 0; r < 4; ++r) {
      const int j = wl * ROWS + jj0 + r, i = j * F3_N + lane, si = j * F3_PITCH + lane;
      const cplx u = cscale(gu[r], s), v = cscale(gv[r], s);
      const cplx Lu = tb[(NS - 1) * TILE + si], Lv = tb[(2 * NS - 1) * TILE + si];
      const cplx q = gq[r], D = gD[r];
      double ha = 0.5 * kp2, hb = 0.5 * kp2;
      if (SYM && kp2 != 0.0) { ha *= gA[r].x; hb *= gA[r].y; }
      cplx Ku, Kv;
      if (SYM) {                                                       // Eq. 40; its +(lap alpha) w / 4 term sits in q
        const cplx Tu = tb[si], Tv = tb[NS * TILE + si];
        Ku = make_double2(-0.25 * (Lu.x + Tu.x) + ha * u.x, -0.25 * (Lu.y + Tu.y) + ha * u.y);
        Kv = make_double2(-0.25 * (Lv.x + Tv.x) + hb * v.x, -0.25 * (Lv.y + Tv.y) + hb * v.y);
      } else {                                                         // Eq. 14
        Ku = make_double2(-0.5 * Lu.x + ha * u.x, -0.5 * Lu.y + ha * u.y);
        Kv = make_double2(-0.5 * Lv.x + hb * v.x, -0.5 * Lv.y + hb * v.y);
      }
      const cplx Hu = cadd(Ku, cadd(cscale(u, q.x), cmul(D, v)));                               // Eqs. 5, 15
      const cplx Hv = csub(cmul(cconj(D), u), cadd(Kv, cscale(v, q.y)));
      e += u.x * Hu.x + u.y * Hu.y + v.x * Hv.x + v.y * Hv.y;
      if (MODE == F3_APPLY) { st_pol_nb(ou + i, Hu, pol.drop); st_pol_nb(ov + i, Hv, pol.drop); }
      else if (MODE == F3_RHS) { st_pol_nb(ou + i, make_double2(Hu.y, -Hu.x), pol.keep); st_pol_nb(ov + i, make_double2(Hv.y, -Hv.x), pol.keep); }   // -i H
      else {
        const cplx c0 = g0[r], c1 = g1[r];
        const cplx xu = make_double2(c0.x + a.kappa * Hu.y, c0.y - a.kappa * Hu.x);             // C_part - i kappa H
        const cplx xv = make_double2(c1.x + a.kappa * Hv.y, c1.y - a.kappa * Hv.x);
        st_pol_nb(ou + i, xu, pol.keep); st_pol_nb(ov + i, xv, pol.keep);
        xx += cabs2(xu) + cabs2(xv);
        xpr += xu.x * u.x + xu.y * u.y + xv.x * v.x + xv.y * v.y;
        xpi += xu.x * u.y - xu.y * u.x + xv.x * v.y - xv.y * v.x;
        pp += cabs2(u) + cabs2(v);
      }
     }
    }
  }
  F3_T(2, 4);
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
template <int MODE, int NT = 128>
__device__ __forceinline__ void f3_body_d(const F3Mega& a, const F3Pol& pol, int g, int id, double* s_eps, double* s_sn) {
  constexpr int PTS = F3_PLANE / F3_DSPLIT / NT;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int ix = id / F3_DSPLIT, half = id - ix * F3_DSPLIT;
  const int cnt = (a.n - g * a.gs < a.gs) ? a.n - g * a.gs : a.gs;
  const size_t M = (size_t)a.NX * F3_PLANE, np = (size_t)a.n * a.NX;
  F3_T0();
  for (int nl = warp; nl < cnt; nl += NT / 32) {
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
  F3_T(3, 0);
  const size_t p0 = (size_t)ix * F3_PLANE + half * (F3_PLANE / F3_DSPLIT) + threadIdx.x;
  const size_t ring = (size_t)(g % F3_RING) * a.gs * 2;
  double acc[PTS][4];
#pragma unroll
  for (int r = 0; r < PTS; ++r) { acc[r][0] = acc[r][1] = acc[r][2] = acc[r][3] = 0.0; }
#pragma unroll 2
  for (int nl = 0; nl < cnt; ++nl) {
    const int n = g * a.gs + nl;
    const double e = s_eps[nl];
    const cplx* Xu = a.X + (ring + 2 * nl) * M + p0;
    const cplx* pu = a.psi + (size_t)(2 * n) * M + p0;
    cplx* ou = a.out + (size_t)(2 * n) * M + p0;
    if (nl + 1 < cnt && (threadIdx.x & 7) == 0) {                 // one request per 128-byte line
#pragma unroll
      for (int r = 0; r < PTS; ++r) {
        f3_pf1(pu + 2 * M + r * NT); f3_pf1(pu + 3 * M + r * NT);
      }
    }
    if (MODE == F3_CORR) {
      const double sP = a.scale ? a.scale[n] : 1.0, ke = a.kappa * e, sn = s_sn[nl];
      const double cp = a.cpref[n], wa = a.w_a[n], wb = a.w_b[n];
      cplx gxu[PTS], gxv[PTS], gpu[PTS], gpv[PTS];          // all loads of this spinor first, then the arithmetic
#pragma unroll
      for (int r = 0; r < PTS; ++r) {
        gxu[r] = __ldcg(Xu + r * NT); gxv[r] = __ldcg(Xu + M + r * NT); gpu[r] = pu[r * NT]; gpv[r] = pu[M + r * NT];
      }
#pragma unroll
      for (int r = 0; r < PTS; ++r) {
        const cplx xu = gxu[r], xv = gxv[r];
        const cplx wu = cscale(gpu[r], sP), wv = cscale(gpv[r], sP);
        const cplx u = make_double2((xu.x - ke * wu.y) * sn, (xu.y + ke * wu.x) * sn);
        const cplx v = make_double2((xv.x - ke * wv.y) * sn, (xv.y + ke * wv.x) * sn);
        st_pol_nb(ou + r * NT, u, pol.drop); st_pol_nb(ou + M + r * NT, v, pol.drop);
        if (a.do_dens) f3_dens_add(acc[r], u, v, cp, wa, wb);
      }
    } else {
      cplx gxu[PTS], gxv[PTS], gpu[PTS], gpv[PTS];
#pragma unroll
      for (int r = 0; r < PTS; ++r) {
        gxu[r] = __ldcg(Xu + r * NT); gxv[r] = __ldcg(Xu + M + r * NT); gpu[r] = pu[r * NT]; gpv[r] = pu[M + r * NT];
      }
#pragma unroll
      for (int r = 0; r < PTS; ++r) {
        const cplx yu = gxu[r], yv = gxv[r];
        const cplx u = gpu[r], v = gpv[r];
        st_pol_nb(ou + r * NT, make_double2(yu.x - e * u.y, yu.y + e * u.x), pol.drop);
        st_pol_nb(ou + M + r * NT, make_double2(yv.x - e * v.y, yv.y + e * v.x), pol.drop);
      }
    }
  }
  F3_T(3, 1);
  if (MODE == F3_CORR && a.do_dens) {
    double* ac = a.acc + (size_t)(g % F3_RING) * 4 * M + p0;
#pragma unroll
    for (int r = 0; r < PTS; ++r)
#pragma unroll
      for (int f = 0; f < 4; ++f) {
        double* q = ac + f * M + r * NT;
        *q = (g < F3_RING ? 0.0 : __ldcg(q)) + acc[r][f];
      }
  }
}

// Cooperative L2 prefetch: every item of tick t fetches its 1/IT share of the read-only inputs the NEXT tick
// will read from HBM -- psi of group t+1 (A items) and C_part of group t-1 (C items of tick t+1) -- so that those
// loads find their lines in L2.  Needs no ticket look-ahead, hence adds no dependency latency.
template <int MODE, int NT = 128>
__device__ __forceinline__ void f3_prefetch_tick(const F3Mega& a, int tick, int r, int chunk, int lines) {
  const size_t M = (size_t)a.NX * F3_PLANE;
  const int lpc = (int)(M * 16 / 128) * 2;                        // 128-byte lines per spinor
  const int q0 = r * chunk + threadIdx.x;
  int q1 = (r + 1) * chunk; if (q1 > lines) q1 = lines;
  const int ga = tick + 1, gc = tick - 1;
  if (ga < a.G) {
    const int rem = a.n - ga * a.gs, lim = (rem < a.gs ? rem : a.gs) * lpc;
    const char* base = (const char*)(a.psi + (size_t)ga * a.gs * 2 * M);
    for (int q = q0; q < q1 && q < lim; q += NT) f3_pf(base + (size_t)q * 128);
  }
  if (MODE == F3_CORR && gc >= 0 && gc < a.G) {
    const int rem = a.n - gc * a.gs, lim = (rem < a.gs ? rem : a.gs) * lpc;
    const char* base = (const char*)(a.cpart + (size_t)gc * a.gs * 2 * M);
    for (int q = q0; q < q1 && q < lim; q += NT) f3_pf(base + (size_t)q * 128);
  }
}

// ---- the persistent kernel ----------------------------------------------------------------------------------
template <bool SYM, int MODE>
__global__ void __launch_bounds__(128, F3_MEGA_OCC) k_f3_mega(F3Mega a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* tiles = reinterpret_cast<cplx*>(smem_raw);
  __shared__ int s_item[2];
  __shared__ double red[4 * F3_NPART];
  __shared__ double s_eps[32], s_sn[32];
  cplx x[F3_N];
  const F3Pol pol = f3_policies();
  const int G = a.G, NX = a.NX;
  int* done = reinterpret_cast<int*>(a.sync + 1);
  const int nA = a.gs * 2 * NX / 4, nB = a.gs * 16, nC = SYM ? a.gs * NX : a.gs * NX / 2;
  const int nD = MODE == F3_APPLY ? 0 : NX * F3_DSPLIT;
  const int IT = nA + nB + nC + nD, total = (G + 3) * IT;
  const int pf_lines = a.gs * 2 * NX * (F3_PLANE * 16 / 128), pf_chunk = (pf_lines + IT - 1) / IT;
  int t1 = 0;
  if (threadIdx.x == 0) t1 = atomicAdd(&a.sync->next, 1);
  for (;;) {
    F3_T0();
    if (threadIdx.x == 0) s_item[0] = t1;
    __syncthreads();
    const int item = s_item[0];
    __syncthreads();
    if (item >= total) break;
    const int tick = item / IT, r = item - tick * IT;
    bool drew = false;
    f3_prefetch_tick<MODE>(a, tick, r, pf_chunk, pf_lines);
    F3_T(4, 0);
    if (r < nA) {
      const int g = tick;
      if (g < G) {
        if (g >= F3_RING) f3_wait(&done[2 * G + g - F3_RING], nC, a.sync);
        F3_T(4, 1);
        f3_body_a<SYM>(a, pol, g, r, tiles, x);
        F3_T0();
        f3_signal(&done[g], &a.sync->next, t1); drew = true;
        F3_T(4, 5);
      }
    } else if (r < nA + nB) {
      const int g = tick - 1;
      if (g >= 0 && g < G) {
        f3_wait(&done[g], nA, a.sync);
        F3_T(4, 2);
        if (NX == 32) f3_body_b<32, SYM>(a, pol, g, r - nA, x);
        else if (NX == 16) f3_body_b<16, SYM>(a, pol, g, r - nA, x);
        else f3_body_b<8, SYM>(a, pol, g, r - nA, x);
        F3_T0();
        f3_signal(&done[G + g], &a.sync->next, t1); drew = true;
        F3_T(4, 5);
      }
    } else if (r < nA + nB + nC) {
      const int g = tick - 2;
      if (g >= 0 && g < G) {
        f3_wait(&done[G + g], nB, a.sync);
        if (MODE != F3_APPLY && g >= F3_RING) f3_wait(&done[3 * G + g - F3_RING], nD, a.sync);
        F3_T(4, 3);
        f3_body_c<SYM, MODE>(a, pol, g, r - nA - nB, tiles, red, x);
        F3_T0();
        f3_signal(&done[2 * G + g], &a.sync->next, t1); drew = true;
        F3_T(4, 5);
      }
    } else {
      const int g = tick - 3;
      if (g >= 0 && g < G) {
        f3_wait(&done[2 * G + g], nC, a.sync);
        if (g >= F3_RING) f3_wait(&done[3 * G + g - F3_RING], nD, a.sync);
        F3_T(4, 4);
        if (MODE != F3_APPLY) f3_body_d<MODE>(a, pol, g, r - nA - nB - nC, s_eps, s_sn);
        F3_T0();
        f3_signal(&done[3 * G + g], &a.sync->next, t1); drew = true;
        F3_T(4, 5);
      }
    }
    if (!drew && threadIdx.x == 0) t1 = atomicAdd(&a.sync->next, 1);
  }
}
