// mega3s.cuh -- the 32^3 stage kernels (Eq. 40 and Eq. 14 operators) with the Laplacian taken axis by axis.
//
// The spectral Laplacian of Eq. 26 is a sum over the axes, lap = d_x^2 + d_y^2 + d_z^2, and each
// term needs transforms along ITS axis only (forward, times -k_d^2 / N_d, inverse on every line of that axis).  So
// no 3-D spectrum has to exist anywhere: the stage is two passes over psi itself instead of the three passes over
// psi / spectrum / spectrum of mega3d.cuh,
//   P (n, x-plane)   : (d_y^2 + d_z^2) of w and of alpha w for both components, one plane per warp, one tile
//                      transposition each way; Q_c = (d_y^2 + d_z^2)(alpha_c w) + alpha_c (d_y^2 + d_z^2) w   -> Q ring
//   XE (n, y-row)    : x-lines in registers (lane = z): d_x^2 w and d_x^2 (alpha w), no shared-memory exchange; then
//                      K_c = -1/4 [ d_x^2(alpha w) + alpha d_x^2 w + Q_c ] + ..., the BdG mix, the eps_n / norm partial
//                      sums and the stage combination along the line                                  -> X ring / H psi
//   D                : unchanged (f3_body_d of mega3d.cuh).
// The same number of line transforms as before (12 per line of a component), but the only intermediate is Q: 1 MB
// per spinor written once and read once, against 2 + 4 + 2 MB of spectrum traffic; three item kinds and two
// dependency levels instead of four and three; 56 instead of 77 items per spinor.  The result differs from the 3-D
// transform only in rounding order.  Ticket dispatch, counters, rings and eviction hints are those of mega3d.cuh.
#pragma once
#include "mega3d.cuh"

// L1-allocating load with an L2 eviction policy
__device__ __forceinline__ cplx ld_ca_pol(const cplx* p, uint64_t pol) {
  cplx v;
  asm volatile("ld.global.ca.L2::cache_hint.v2.f64 {%0, %1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(pol));
  return v;
}

struct F3SMega {
  F3Mega m;                      // spec0 = Q ring [R][gs][2][M]; spec1 unused
  int pm, em;                    // x-planes per P item (1, 2, 4, 8), row pairs per XE item (1, 2, 4)
  double k2zy[64];               // k_z^2 (0..31) then k_y^2 (32..63), natural order (kernel parameters: constant bank)
};

// second derivative along the register index: x <- s * IFFT( -k2[j] / 32 * FFT(x) ); the inverse is conj(FFT(conj .)).
// The spinor's scale s rides on the k-space factor and the closing conjugation is a sign-bit flip (no FP64 issue slot).
__device__ __forceinline__ double f3s_flip(double v) { return __hiloint2double(__double2hiint(v) ^ (int)0x80000000u, __double2loint(v)); }
template <class K2>
__device__ __forceinline__ void f3s_d2(cplx* x, K2 k2, double s) {
  const double sm = -0.03125 * s;
#pragma unroll 1
  for (int dir = 0; dir < 2; ++dir) {
    fft_reg<F3_N, false>(x);
    if (dir == 0) {
#pragma unroll
      for (int j = 0; j < F3_N; ++j) {
        const double f = k2(j) * sm;
        x[j] = make_double2(x[j].x * f, -x[j].y * f);
      }
    }
  }
#pragma unroll
  for (int j = 0; j < F3_N; ++j) x[j].y = f3s_flip(x[j].y);
}

// ---- P: (d_y^2 + d_z^2) of the four fields u, alpha_a u, v, alpha_b v of one (spinor, x-plane), one per warp -----
// Eq. 14 (SYM = false): the item is two x-planes, one (plane, component) per warp, Q_c = (d_y^2 + d_z^2) w, no pairing.
template <bool SYM>
__device__ __forceinline__ void f3s_body_p(const F3SMega& A, const F3Pol& pol, int g, int ip, cplx* tiles, cplx* x) {
  const F3Mega& a = A.m;
  constexpr int TILE = F3_N * F3_PITCH, PER = SYM ? F3_N : F3_N / 2;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nl = ip / PER, rr = ip - nl * PER, ix = SYM ? rr : 2 * rr + (warp >> 1), n = g * a.gs + nl;
  const bool valid = n < a.n;
  const int c = SYM ? warp >> 1 : warp & 1, t = SYM ? warp & 1 : 0;   // t = 0: w (times alpha afterwards), t = 1: alpha w
  const size_t M = (size_t)F3_N * F3_PLANE, pl = (size_t)ix * F3_PLANE;
  cplx* S = tiles + warp * TILE;
  F3_T0();
  if (valid) {
    const cplx* src = a.psi + (size_t)(2 * n + c) * M + pl;
    const double* al = a.F.alpha[c] + pl;
    const double s = a.scale ? a.scale[n] : 1.0;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
      if (SYM && t) {
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = cscale(ld_ca_pol(src + j * F3_N + lane, pol.keep), al[j * F3_N + lane]);
      } else {
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = ld_ca_pol(src + j * F3_N + lane, pol.keep);   // (y = j, z = lane); the second pass hits L1 / L2; XE and D re-read it
      }
      if (pass == 0) F3_T(0, 0); else F3_T(0, 2);
      if (pass == 0) {                                          // z-lines: transpose, differentiate, transpose back
#pragma unroll
        for (int j = 0; j < F3_N; ++j) S[j * F3_PITCH + lane] = x[j];
        __syncwarp();
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = S[lane * F3_PITCH + j];
      }
      f3s_d2(x, [&](int j) { return A.k2zy[pass * 32 + j]; }, s);
      if (pass == 0) F3_T(0, 1); else F3_T(0, 3);
      if (pass == 0) {
#pragma unroll
        for (int j = 0; j < F3_N; ++j) S[lane * F3_PITCH + j] = x[j];
        __syncwarp();
      }
    }
    if (!SYM) {                                                 // straight to the Q ring: nothing to pair with
      cplx* q = a.spec0 + (((size_t)(g % F3_RING) * a.gs + nl) * 2 + c) * M + pl;
#pragma unroll
      for (int j = 0; j < F3_N; ++j) st_pol(q + j * F3_N + lane, cadd(x[j], S[j * F3_PITCH + lane]), pol.keep);
      __syncwarp();
      return;
    }
#pragma unroll
    for (int j = 0; j < F3_N; ++j) {
      const cplx z = S[j * F3_PITCH + lane];
      const double f = t ? 1.0 : al[j * F3_N + lane];
      S[j * F3_PITCH + lane] = make_double2((x[j].x + z.x) * f, (x[j].y + z.y) * f);
    }
  }
  if (!SYM) return;
  F3_T(0, 4);
  if (c == 0) asm volatile("bar.sync 1, 64;" ::: "memory"); else asm volatile("bar.sync 2, 64;" ::: "memory");   // the pair (w, alpha w)
  F3_T(0, 5);
  if (valid) {                                                  // Q_c = alpha (d_y^2 + d_z^2) w + (d_y^2 + d_z^2)(alpha w)
    cplx* q = a.spec0 + (((size_t)(g % F3_RING) * a.gs + nl) * 2 + c) * M + pl;
    const cplx* T0 = tiles + (2 * c) * TILE;
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      const int j = 16 * t + r, si = j * F3_PITCH + lane;
      st_pol(q + j * F3_N + lane, cadd(T0[si], T0[TILE + si]), pol.keep);
    }
  }
  if (c == 0) asm volatile("bar.sync 1, 64;" ::: "memory"); else asm volatile("bar.sync 2, 64;" ::: "memory");   // tiles free again
  F3_T(0, 6);
}

struct F3SRow { cplx u, v, D, q, Qu, Qv, cu, cv; double Aa, Ab; };   // the epilogue inputs of one lattice point

// ---- XE: the x-lines of one (spinor, y-row) by a PAIR of warps (lane = z): warp c of the pair differentiates
// component c (alpha d_x^2 w + d_x^2(alpha w), parked in shared memory); after a pair barrier each warp finishes half of
// the line for BOTH components, so that psi, the fields, Q and C_part are read once per point ---------------------------
template <bool SYM, int MODE>
__device__ __forceinline__ void f3s_body_xe(const F3SMega& A, const F3Pol& pol, int g, int ie, cplx* park, double* red, cplx* x) {
  const F3Mega& a = A.m;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int pr = warp >> 1, c = warp & 1;
  const int nl = ie >> 4, y = 2 * (ie & 15) + pr, n = g * a.gs + nl;
  if (n >= a.n) return;                                         // the whole CTA (one spinor per item)
  const size_t M = (size_t)F3_N * F3_PLANE, off = (size_t)y * F3_N + lane;     // point (x = j): off + j * F3_PLANE
  const size_t ring = ((size_t)(g % F3_RING) * a.gs + nl) * 2;
  const double s = a.scale ? a.scale[n] : 1.0, kp2 = a.kperp2[n];
  const cplx* pu = a.psi + (size_t)(2 * n) * M + off;
  const cplx* pv = pu + M;
  const cplx* pk = a.pack + off;
  cplx* P = park + threadIdx.x;                                 // this thread's slots P[j * 128]
  const cplx* Pu = park + (pr * 64 + lane);                     // the pair's parked lines of u and v
  const cplx* Pv = Pu + 32;
  F3_T0();
  {
    const cplx* pc = c ? pv : pu;
    const double* al = a.F.alpha[c] + off;
#pragma unroll 1
    for (int t = 0; t < (SYM ? 2 : 1); ++t) {                   // t = 0: alpha d_x^2 w (Eq. 14: d_x^2 w), t = 1: d_x^2 (alpha w)
      if (t) {
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = cscale(pc[(size_t)j * F3_PLANE], al[(size_t)j * F3_PLANE]);
      } else {
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = pc[(size_t)j * F3_PLANE];
      }
      F3_T(1, 0);
      f3s_d2(x, [&](int j) { return a.kx2[j]; }, s);
      F3_T(1, 1);
      if (t == 0) {
#pragma unroll
        for (int j = 0; j < F3_N; ++j) P[j * 128] = SYM ? cscale(x[j], al[(size_t)j * F3_PLANE]) : x[j];
      } else {
#pragma unroll
        for (int j = 0; j < F3_N; ++j) { const cplx z = P[j * 128]; P[j * 128] = cadd(x[j], z); }
      }
    }
  }
  F3_T(1, 2);
  if (pr == 0) asm volatile("bar.sync 1, 64;" ::: "memory"); else asm volatile("bar.sync 2, 64;" ::: "memory");
  F3_T(1, 4);
  double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
  {
    const cplx* Qu = a.spec0 + ring * M + off;
    const cplx* cu = a.cpart + (size_t)(2 * n) * M + off;
    cplx* ou = (MODE == F3_APPLY ? a.out + (size_t)(2 * n) * M : a.X + ring * M) + off;
    // two points per batch, two batches in flight: the loads of the next batch are issued before the arithmetic
    // (and the stores) of the current one
    auto load = [&](F3SRow* b, int j0) {
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        const size_t i = (size_t)(j0 + r) * F3_PLANE;
        b[r].u = pu[i]; b[r].v = pv[i]; b[r].q = pk[i]; b[r].D = pk[M + i];
        if (SYM && kp2 != 0.0) { const cplx t = pk[2 * M + i]; b[r].Aa = t.x; b[r].Ab = t.y; } else { b[r].Aa = b[r].Ab = 0.0; }
        b[r].Qu = ld_pol(Qu + i, pol.drop); b[r].Qv = ld_pol(Qu + M + i, pol.drop);    // last use of Q
        if (MODE == F3_CORR) { b[r].cu = ld_pol(cu + i, pol.drop); b[r].cv = ld_pol(cu + M + i, pol.drop); }   // read once
      }
    };
    auto comp = [&](const F3SRow* b, int j0) {
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        const size_t i = (size_t)(j0 + r) * F3_PLANE;
        const cplx u = cscale(b[r].u, s), v = cscale(b[r].v, s);
        const cplx Lu = cadd(Pu[(j0 + r) * 128], b[r].Qu), Lv = cadd(Pv[(j0 + r) * 128], b[r].Qv);
        const double ha = SYM ? 0.5 * kp2 * b[r].Aa : 0.5 * kp2, hb = SYM ? 0.5 * kp2 * b[r].Ab : 0.5 * kp2;
        constexpr double kf = SYM ? -0.25 : -0.5;                                           // Eq. 40 (its +(lap alpha) w / 4 sits in q) | Eq. 14
        const cplx Ku = make_double2(kf * Lu.x + ha * u.x, kf * Lu.y + ha * u.y);
        const cplx Kv = make_double2(kf * Lv.x + hb * v.x, kf * Lv.y + hb * v.y);
        const cplx D = b[r].D;
        const cplx Hu = cadd(Ku, cadd(cscale(u, b[r].q.x), cmul(D, v)));                  // Eqs. 5, 15
        const cplx Hv = csub(cmul(cconj(D), u), cadd(Kv, cscale(v, b[r].q.y)));
        e += u.x * Hu.x + u.y * Hu.y + v.x * Hv.x + v.y * Hv.y;
        if (MODE == F3_APPLY) { st_pol_nb(ou + i, Hu, pol.drop); st_pol_nb(ou + M + i, Hv, pol.drop); }
        else if (MODE == F3_RHS) {                                                         // -i H
          st_pol_nb(ou + i, make_double2(Hu.y, -Hu.x), pol.keep); st_pol_nb(ou + M + i, make_double2(Hv.y, -Hv.x), pol.keep);
        } else {
          const cplx xu = make_double2(b[r].cu.x + a.kappa * Hu.y, b[r].cu.y - a.kappa * Hu.x);   // C_part - i kappa H
          const cplx xv = make_double2(b[r].cv.x + a.kappa * Hv.y, b[r].cv.y - a.kappa * Hv.x);
          st_pol_nb(ou + i, xu, pol.keep); st_pol_nb(ou + M + i, xv, pol.keep);
          xx += cabs2(xu) + cabs2(xv);
          xpr += xu.x * u.x + xu.y * u.y + xv.x * v.x + xv.y * v.y;
          xpi += xu.x * u.y - xu.y * u.x + xv.x * v.y - xv.y * v.x;
          pp += cabs2(u) + cabs2(v);
        }
      }
    };
    F3SRow b0[2], b1[2];
    const int jb = 16 * c;                                      // this warp's half of the line
    load(b0, jb);
#pragma unroll 1
    for (int j0 = jb; j0 < jb + 16; j0 += 4) {
      load(b1, j0 + 2);
      comp(b0, j0);
      if (j0 + 4 < jb + 16) load(b0, j0 + 4);
      comp(b1, j0 + 2);
    }
  }
  F3_T(1, 3);
  e = warp_sum(e);
  if (MODE == F3_CORR) { xx = warp_sum(xx); xpr = warp_sum(xpr); xpi = warp_sum(xpi); pp = warp_sum(pp); }
  if (c == 1 && lane == 0) {
    double* q = red + pr * F3_NPART;
    q[0] = e;
    if (MODE == F3_CORR) { q[1] = xx; q[2] = xpr; q[3] = xpi; q[4] = pp; }
  }
  if (pr == 0) asm volatile("bar.sync 1, 64;" ::: "memory"); else asm volatile("bar.sync 2, 64;" ::: "memory");
  if (c == 0 && lane == 0) {
    const double* q = red + pr * F3_NPART;
    const size_t np = (size_t)a.n * F3_N, o = (size_t)n * F3_N + y;
    a.part[o] = e + q[0];
    if (MODE == F3_CORR) { a.part[np + o] = xx + q[1]; a.part[2 * np + o] = xpr + q[2]; a.part[3 * np + o] = xpi + q[3]; a.part[4 * np + o] = pp + q[4]; }
  }
}

// tick t: P(t), XE(t-1), D(t-2).  done[0..G) P, [G..2G) XE, [2G..3G) D.
#ifndef F3S_OCC
#define F3S_OCC F3_MEGA_OCC
#endif
template <bool SYM, int MODE>
__global__ void __launch_bounds__(128, F3S_OCC) k_f3s_mega(F3SMega A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* tiles = reinterpret_cast<cplx*>(smem_raw);
  __shared__ int s_item[2];
  __shared__ double s_eps[32], s_sn[32], red[2 * F3_NPART];
  const F3Mega& a = A.m;
  cplx x[F3_N];
  const F3Pol pol = f3_policies();
  const int G = a.G;
  int* done = reinterpret_cast<int*>(a.sync + 1);
  const int nP = a.gs * (SYM ? F3_N : F3_N / 2) / A.pm, nE = a.gs * 16 / A.em, nD = MODE == F3_APPLY ? 0 : F3_N * F3_DSPLIT;
  const int IT = nP + nE + nD, total = (G + 2) * IT;
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
    F3_T(4, 0);
    F3_T(4, 6);
    if (r < nP) {
      const int g = tick;
      if (g < G) {
        if (g >= F3_RING) f3_wait(&done[G + g - F3_RING], nE, a.sync);                 // the Q slot is free
        F3_T(4, 1);
        for (int k = 0; k < A.pm; ++k) { f3s_body_p<SYM>(A, pol, g, r * A.pm + k, tiles, x); }
        F3_T0();
        f3_signal(&done[g], &a.sync->next, t1); drew = true;
        F3_T(4, 5);
      }
    } else if (r < nP + nE) {
      const int g = tick - 1;
      if (g >= 0 && g < G) {
        f3_wait(&done[g], nP, a.sync);
        if (MODE != F3_APPLY && g >= F3_RING) f3_wait(&done[2 * G + g - F3_RING], nD, a.sync);   // the X slot is free
        F3_T(4, 2);
        for (int k = 0; k < A.em; ++k) { if (k) __syncthreads(); f3s_body_xe<SYM, MODE>(A, pol, g, (r - nP) * A.em + k, tiles, red, x); }
        F3_T0();
        f3_signal(&done[G + g], &a.sync->next, t1); drew = true;
        F3_T(4, 5);
      }
    } else {
      const int g = tick - 2;
      if (g >= 0 && g < G) {
        f3_wait(&done[G + g], nE, a.sync);
        if (g >= F3_RING) f3_wait(&done[2 * G + g - F3_RING], nD, a.sync);             // the density slot
        F3_T(4, 4);
        if (MODE != F3_APPLY) f3_body_d<MODE>(a, pol, g, r - nP - nE, s_eps, s_sn);
        F3_T0();
        f3_signal(&done[2 * G + g], &a.sync->next, t1); drew = true;
        F3_T(4, 5);
      }
    }
    if (!drew && threadIdx.x == 0) t1 = atomicAdd(&a.sync->next, 1);
  }
}
