// density.cuh -- density accumulation (Eqs. 7a-g; 29b-e, 30b-e) and the pointwise
// functional (Eqs. 9-12, 19-22 PAPER.md:195-255, 311-337).
#pragma once
#include "common.cuh"

// raw density planes, each M doubles
enum { DP_RHO_A = 0, DP_RHO_B, DP_NU_RE, DP_NU_IM, DP_TAU_A, DP_TAU_B, DP_JA0, DP_JA1, DP_JA2, DP_JB0, DP_JB1, DP_JB2, DP_BP_RE, DP_BP_IM, DP_COUNT };

struct DensArgs {
  const cplx* psi;                       // chunk base
  const double *scale, *cpref, *kperp2, *w_a, *w_b;   // per spinor of the chunk (scale nullable)
  const cplx* grad[3];                   // d_j psi (already scaled), [2 n + c][M]; null when not needed
  const cplx* lap;                       // lap psi (already scaled), same layout; for B' of Eq. 68 (mask WSLDA_D_BP)
  int nd;
  int64_t M, n_count, per_group;
  unsigned mask;                         // WSLDA_D_* bits
};

// grid (ceil(M / threads), G): each thread owns one lattice point and sums the spinors of its group in
// increasing n; partial planes go to part[g][DP_COUNT][M].  No atomics: bit-reproducible run to run.
__global__ void __launch_bounds__(WS_PT_THREADS) k_density(DensArgs a, double* part) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.M) return;
  const int64_t n0 = (int64_t)blockIdx.y * a.per_group;
  const int64_t n1 = (n0 + a.per_group < a.n_count) ? n0 + a.per_group : a.n_count;
  const bool need_g = (a.mask & (WSLDA_D_TAU | WSLDA_D_J)) != 0;
  double acc[DP_COUNT];
#pragma unroll
  for (int f = 0; f < DP_COUNT; ++f) acc[f] = 0.0;
  for (int64_t n = n0; n < n1; ++n) {
    const double s = a.scale ? a.scale[n] : 1.0;
    const cplx u = cscale(a.psi[2 * n * a.M + i], s), v = cscale(a.psi[(2 * n + 1) * a.M + i], s);
    const double cp = a.cpref[n], cwa = cp * a.w_a[n], cwb = cp * a.w_b[n];
    const double u2 = cabs2(u), v2 = cabs2(v);
    acc[DP_RHO_A] += cwa * u2;                                               // Eq. 7a
    acc[DP_RHO_B] += cwb * v2;                                               // Eq. 7b
    const double wn = 0.5 * cp * (a.w_b[n] - a.w_a[n]);                      // Eq. 7e: u v^*
    acc[DP_NU_RE] += wn * (u.x * v.x + u.y * v.y);
    acc[DP_NU_IM] += wn * (u.y * v.x - u.x * v.y);
    if (need_g) {
      double gu2 = 0.0, gv2 = 0.0;
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if (d < a.nd) {
          const cplx gu = a.grad[d][2 * n * a.M + i], gv = a.grad[d][(2 * n + 1) * a.M + i];
          gu2 += cabs2(gu); gv2 += cabs2(gv);
          acc[DP_JA0 + d] += -cwa * (u.y * gu.x - u.x * gu.y);               // Eq. 7f: -Im[u grad u^*]
          acc[DP_JB0 + d] += cwb * (v.y * gv.x - v.x * gv.y);                // Eq. 7g: +Im[v grad v^*]
        }
      }
      acc[DP_TAU_A] += cwa * (gu2 + a.kperp2[n] * u2);                        // Eqs. 7c, 29c, 30c
      acc[DP_TAU_B] += cwb * (gv2 + a.kperp2[n] * v2);                        // Eq. 7d
    }
    if (a.mask & WSLDA_D_BP) {                                                // Eq. 68; lap -> lap - k_perp^2 for a plane-wave factor
      const cplx lu = a.lap[2 * n * a.M + i], lv = a.lap[(2 * n + 1) * a.M + i];
      const cplx Lu = make_double2(lu.x - a.kperp2[n] * u.x, lu.y - a.kperp2[n] * u.y);
      const cplx Lv = make_double2(lv.x - a.kperp2[n] * v.x, lv.y - a.kperp2[n] * v.y);
      const cplx t = cadd(cmul(u, cconj(Lv)), cmul(cconj(v), Lu));
      acc[DP_BP_RE] += -0.5 * wn * t.x; acc[DP_BP_IM] += -0.5 * wn * t.y;
    }
  }
  double* p = part + (int64_t)blockIdx.y * DP_COUNT * a.M + i;
#pragma unroll
  for (int f = 0; f < DP_COUNT; ++f) p[f * a.M] = acc[f];
}

__device__ __host__ inline unsigned plane_bit(int f) {
  return (f <= DP_RHO_B) ? WSLDA_D_RHO : (f <= DP_NU_IM) ? WSLDA_D_NU : (f <= DP_TAU_B) ? WSLDA_D_TAU : (f <= DP_JB2) ? WSLDA_D_J : WSLDA_D_BP;
}

// raw[f][i] = (accumulate ? raw[f][i] : 0) + sum_g part[g][f][i], groups in increasing order
__global__ void k_density_reduce(const double* part, int G, double* raw, int64_t M, unsigned mask, int accumulate) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int f = blockIdx.y;
  if (i >= M || !(mask & plane_bit(f))) return;
  double s = accumulate ? raw[f * M + i] : 0.0;
  for (int g = 0; g < G; ++g) s += part[((int64_t)g * DP_COUNT + f) * M + i];
  raw[f * M + i] = s;
}

struct FuncParams {
  int func_id, force_a1, spin_symmetric, current_terms, quantum_friction;
  double qf_alpha, qf_beta, qf_gamma, qf_rho0, qf_nreq;
  double four_pi_as, C, E_cut, rho_floor, mu_a, mu_b;
};

// densities as the functional sees them: folded per Eq. 8 when spin_symmetric
__device__ inline void folded(const double* raw, int64_t M, int64_t i, int sym, double& ra, double& rb, double& ta,
                              double& tb, cplx& nu) {
  ra = raw[DP_RHO_A * M + i]; rb = raw[DP_RHO_B * M + i];
  ta = raw[DP_TAU_A * M + i]; tb = raw[DP_TAU_B * M + i];
  nu = make_double2(raw[DP_NU_RE * M + i], raw[DP_NU_IM * M + i]);
  if (sym) { ra = rb = ra + rb; ta = tb = ta + tb; nu = cscale(nu, 2.0); }
}

__device__ inline double aslda_A(double p) {      // Eq. 12a
  const double p2 = p * p;
  return 1.094 + 0.156 * p * (1.0 - 2.0 * p2 / 3.0 + p2 * p2 / 5.0) - 0.532 * p2 * (1.0 - p2 + p2 * p2 / 3.0);
}
__device__ inline double aslda_dA(double p) { const double q = 1.0 - p * p; return q * q * (0.156 - 1.064 * p); }

// Regulariser Lambda_c, Eqs. 20-21; k0^2 <= 0 by analytic continuation (R5).
__device__ inline double lambda_c(double alpha_p, double V_p, double mu_p, double E_c, bool& empty) {
  const double PI = 3.14159265358979323846;
  const double k02 = 2.0 * (mu_p - V_p) / alpha_p, kc2 = 2.0 * (E_c + mu_p - V_p) / alpha_p;
  empty = false;
  if (kc2 <= 0.0) { empty = true; return 0.0; }
  const double kc = sqrt(kc2), pref = kc / (2.0 * PI * PI * alpha_p);
  if (k02 > 0.0) {
    const double k0 = sqrt(k02);
    return pref * (1.0 - k0 / (2.0 * kc) * log((kc + k0) / (kc - k0)));
  }
  const double kap = sqrt(-k02);
  if (kap == 0.0) return pref;
  return pref * (1.0 - kap / kc * atan(kc / kap));
}

// One thread per lattice point: alpha_sigma, V_sigma, U_sigma, Lambda_c, g_eff, Delta = -g_eff nu (Eq. 10).
// With current_terms: A_sigma = dE/dj_sigma = (1 - alpha_sigma) j_sigma / rho_sigma (Eqs. 9b-c)
// into cur_A [2][3][M], W_sigma = A_sigma - v_ext_sigma into cur_W, and the j-terms of V_sigma.
__global__ void k_potentials(FuncParams P, const double* raw, const double* vext_a, const double* vext_b, int use_frozen,
                             double* alpha_a, double* alpha_b, double* V_a, double* V_b, double* U_a, double* U_b,
                             double* lambda, double* geff, cplx* delta, int64_t M, double* cur_A, const double* cur_v,
                             double* cur_W) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  const double PI = 3.14159265358979323846;
  double ra, rb, ta, tb; cplx nu;
  folded(raw, M, i, P.spin_symmetric, ra, rb, ta, tb, nu);
  double rho = ra + rb; if (rho < P.rho_floor) rho = P.rho_floor;
  double aa = 1.0, ab = 1.0, Va0 = 0.0, Vb0 = 0.0, inv_g0;
  if (P.func_id == WSLDA_FUNC_BDG) {
    inv_g0 = 1.0 / P.four_pi_as;                               // Eq. 11
  } else {
    double p = (ra - rb) / rho; p = fmin(1.0, fmax(-1.0, p));
    double dAp = 0.0, dAm = 0.0;
    if (!P.force_a1) { aa = aslda_A(p); ab = aslda_A(-p); dAp = aslda_dA(p); dAm = aslda_dA(-p); }
    const double sp = 0.5 * (1.0 + p), sm = 0.5 * (1.0 - p), c23 = cbrt(4.0);
    const double sp23 = cbrt(sp * sp), sm23 = cbrt(sm * sm), sp53 = sp * sp23, sm53 = sm * sm23;
    const double B = c23 * (0.357 + 0.642 * p * p - aa * sp53 - ab * sm53);                        // Eq. 12b
    const double dB = c23 * (1.284 * p - dAp * sp53 - (5.0 / 6.0) * aa * sp23 + dAm * sm53 + (5.0 / 6.0) * ab * sm23);
    const double x = cbrt(3.0 * PI * PI * rho), eF = 0.5 * x * x;                                  // Eq. 9d
    const double dp_a = 2.0 * rb / (rho * rho), dp_b = -2.0 * ra / (rho * rho);
    const double common = 0.5 * dAp * ta - 0.5 * dAm * tb + 0.6 * rho * eF * dB;
    Va0 = common * dp_a + B * eF;
    Vb0 = common * dp_b + B * eF;
    inv_g0 = cbrt(rho) / P.C;                                  // Eq. 19 in reading R1
    if (P.current_terms) {                                     // energy density + sum (1 - alpha) j^2 / (2 rho_sigma)
      double ja[3], jb[3], ja2 = 0.0, jb2 = 0.0;
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const double a = raw[(DP_JA0 + d) * M + i], b = raw[(DP_JB0 + d) * M + i];
        ja[d] = P.spin_symmetric ? a + b : a; jb[d] = P.spin_symmetric ? a + b : b;
        ja2 += ja[d] * ja[d]; jb2 += jb[d] * jb[d];
      }
      const double rsa = ra < P.rho_floor ? P.rho_floor : ra, rsb = rb < P.rho_floor ? P.rho_floor : rb;
#pragma unroll
      for (int d = 0; d < 3; ++d) { cur_A[d * M + i] = (1.0 - aa) * ja[d] / rsa; cur_A[(3 + d) * M + i] = (1.0 - ab) * jb[d] / rsb; }
      const double dal = -0.5 * dAp * ja2 / rsa + 0.5 * dAm * jb2 / rsb;
      Va0 += dal * dp_a - 0.5 * (1.0 - aa) * ja2 / (rsa * rsa);
      Vb0 += dal * dp_b - 0.5 * (1.0 - ab) * jb2 / (rsb * rsb);
    }
  }
  if (P.current_terms) {
#pragma unroll
    for (int d = 0; d < 6; ++d) {
      const double A = P.func_id == WSLDA_FUNC_BDG ? 0.0 : cur_A[d * M + i];
      if (P.func_id == WSLDA_FUNC_BDG) cur_A[d * M + i] = 0.0;
      cur_W[d * M + i] = A - cur_v[d * M + i];
    }
  }
  bool empty = false;
  const double va = vext_a[i], vb = vext_b[i];
  const double lam = use_frozen ? lambda[i]
                                : lambda_c(0.5 * (aa + ab), 0.5 * (Va0 + va + Vb0 + vb), 0.5 * (P.mu_a + P.mu_b), P.E_cut, empty);
  const double g = empty ? 0.0 : 1.0 / (inv_g0 - lam);
  const cplx D = make_double2(-g * nu.x, -g * nu.y);            // Eq. 10
  double Va = Va0, Vb = Vb0;
  if (P.func_id == WSLDA_FUNC_ASLDA) {
    const double r13 = cbrt(rho), t = cabs2(D) / (3.0 * P.C * r13 * r13);
    Va -= t; Vb -= t;
  }
  alpha_a[i] = aa; alpha_b[i] = ab; V_a[i] = Va; V_b[i] = Vb; U_a[i] = Va + va; U_b[i] = Vb + vb;
  lambda[i] = lam; geff[i] = g; delta[i] = D;
}

// same sums for many groups (small lattices: G ~ 1000): one warp per (plane, point), lanes stride over the groups and
// finish with the fixed shuffle tree -- still deterministic, G-fold more parallel.  grid (ceil(M / 8), DP_COUNT) x 256
__global__ void k_density_reduce_wide(const double* part, int G, double* raw, int64_t M, unsigned mask, int accumulate) {
  const int64_t i = (int64_t)blockIdx.x * 8 + (threadIdx.x >> 5);
  const int f = blockIdx.y, lane = threadIdx.x & 31;
  if (i >= M || !(mask & plane_bit(f))) return;
  double s = 0.0;
  for (int g = lane; g < G; g += 32) s += part[((int64_t)g * DP_COUNT + f) * M + i];
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) raw[f * M + i] = (accumulate ? raw[f * M + i] : 0.0) + s;
}

// folded density field for wslda_get_field
__global__ void k_get_density(const double* raw, int64_t M, int sym, int field_id, double* dst) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  double ra, rb, ta, tb; cplx nu;
  folded(raw, M, i, sym, ra, rb, ta, tb, nu);
  switch (field_id) {
    case WSLDA_F_RHO_A: dst[i] = ra; break;
    case WSLDA_F_RHO_B: dst[i] = rb; break;
    case WSLDA_F_TAU_A: dst[i] = ta; break;
    case WSLDA_F_TAU_B: dst[i] = tb; break;
    case WSLDA_F_NU: dst[2 * i] = nu.x; dst[2 * i + 1] = nu.y; break;
    case WSLDA_F_BP: { const double f2 = sym ? 2.0 : 1.0; dst[2 * i] = f2 * raw[DP_BP_RE * M + i]; dst[2 * i + 1] = f2 * raw[DP_BP_IM * M + i]; } break;
    default: {
      const bool is_a = field_id <= WSLDA_F_JA_Z;
      const int d = is_a ? field_id - WSLDA_F_JA_X : field_id - WSLDA_F_JB_X;
      const double ja = raw[(DP_JA0 + d) * M + i], jb = raw[(DP_JB0 + d) * M + i];
      dst[i] = sym ? ja + jb : (is_a ? ja : jb);
    }
  }
}

// ---- observables (Eqs. 33a-g): particle numbers and the energy terms from the current density block
// and potentials.  One thread per lattice point, fixed-order block sums -> epart[block][WS_NOBS]; k_energy_final adds the
// blocks in index order (bit-reproducible) and, given a reference, runs the conservation check of the time-dependent
// codes: |N_sigma - N_ref| <= tol_n N_ref and |E - E_ref| <= tol_e |E_ref|, else *flag = 1.
#define WS_NOBS 10      // N_a N_b E_kin E_pot E_pair E_pot_ext E_pair_ext E_total E_curr E_vel_ext
struct ObsArgs {
  FuncParams P;
  const double *raw, *alpha_a, *alpha_b, *vext_a, *vext_b, *cur_v;
  const cplx *delta, *dext;
  double dVf;           // dV * L_perp
  int64_t M;
};
__global__ void __launch_bounds__(256) k_energy(ObsArgs a, double* epart) {
  __shared__ double sh[32];
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, M = a.M;
  double v[WS_NOBS];
#pragma unroll
  for (int q = 0; q < WS_NOBS; ++q) v[q] = 0.0;
  if (i < M) {
    const double PI = 3.14159265358979323846;
    double ra, rb, ta, tb; cplx nu;
    folded(a.raw, M, i, a.P.spin_symmetric, ra, rb, ta, tb, nu);
    const double aa = a.alpha_a[i], ab = a.alpha_b[i];
    v[0] = ra; v[1] = rb;
    v[2] = 0.5 * (aa * ta + ab * tb);                                                      // 33a
    if (a.P.func_id == WSLDA_FUNC_ASLDA) {
      double rho = ra + rb; if (rho < a.P.rho_floor) rho = a.P.rho_floor;
      double p = (ra - rb) / rho; p = fmin(1.0, fmax(-1.0, p));
      const double sp = 0.5 * (1.0 + p), sm = 0.5 * (1.0 - p);
      const double B = cbrt(4.0) * (0.357 + 0.642 * p * p - aa * sp * cbrt(sp * sp) - ab * sm * cbrt(sm * sm));
      const double x = cbrt(3.0 * PI * PI * rho);
      v[3] = 0.6 * B * rho * 0.5 * x * x;                                                  // 33b
    }
    const cplx D = a.delta[i], De = a.dext[i];
    v[4] = -(D.x * nu.x + D.y * nu.y);                                                     // 33c: -Re(conj(Delta) nu)
    v[5] = a.vext_a[i] * ra + a.vext_b[i] * rb;                                            // 33e
    v[6] = -2.0 * (De.x * nu.x + De.y * nu.y);                                             // 33f: -(Delta_ext nu^* + h.c.)
    if (a.P.current_terms) {
      double ja2 = 0.0, jb2 = 0.0, vj = 0.0;
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const double x = a.raw[(DP_JA0 + d) * M + i], y = a.raw[(DP_JB0 + d) * M + i];
        const double ja = a.P.spin_symmetric ? x + y : x, jb = a.P.spin_symmetric ? x + y : y;
        ja2 += ja * ja; jb2 += jb * jb;
        vj += a.cur_v[d * M + i] * ja + a.cur_v[(3 + d) * M + i] * jb;
      }
      const double rsa = ra < a.P.rho_floor ? a.P.rho_floor : ra, rsb = rb < a.P.rho_floor ? a.P.rho_floor : rb;
      v[2] -= 0.5 * (aa * ja2 / rsa + ab * jb2 / rsb);                                     // 33a, the -j^2/rho part
      v[8] = 0.5 * (ja2 / rsa + jb2 / rsb);                                                // 33d
      v[9] = -vj;                                                                          // 33g
    }
  }
#pragma unroll
  for (int q = 0; q < WS_NOBS; ++q) {
    if (q == 7) continue;
    const double r = block_sum(v[q], sh);
    if (threadIdx.x == 0) epart[(int64_t)blockIdx.x * WS_NOBS + q] = r * a.dVf;
  }
}
__global__ void k_energy_final(const double* epart, int nblk, double* out, const double* ref, double tol_n, double tol_e, int* flag) {
  if (threadIdx.x || blockIdx.x) return;
  double s[WS_NOBS];
  for (int q = 0; q < WS_NOBS; ++q) s[q] = 0.0;
  for (int b = 0; b < nblk; ++b)
    for (int q = 0; q < WS_NOBS; ++q) if (q != 7) s[q] += epart[(int64_t)b * WS_NOBS + q];
  s[7] = s[2] + s[3] + s[4] + s[5] + s[6] + s[8] + s[9];
  for (int q = 0; q < WS_NOBS; ++q) out[q] = s[q];
  if (ref && flag) {
    bool bad = !(s[7] == s[7]);                                                            // NaN
    for (int q = 0; q < 2; ++q) bad = bad || fabs(s[q] - ref[q]) > tol_n * fabs(ref[q]);
    bad = bad || fabs(s[7] - ref[7]) > tol_e * fabs(ref[7]);
    if (bad) *flag = 1;
  }
}

// ---- quantum friction (Eqs. 66-70), applied after k_potentials: divj[2][M] = div j_sigma (spectral),
// obs = the observables of k_energy_final (N_a, N_b in obs[0], obs[1]) -----------------------------------------------------
__global__ void k_qf(FuncParams P, const double* raw, const double* divj, const double* obs, double* V_a, double* V_b, double* U_a,
                     double* U_b, cplx* delta, int64_t M) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  const double va = -P.qf_alpha / P.qf_rho0 * divj[i], vb = -P.qf_alpha / P.qf_rho0 * divj[M + i];          // Eq. 66
  V_a[i] += va; U_a[i] += va; V_b[i] += vb; U_b[i] += vb;
  const double gt = P.qf_gamma * ((obs[0] + obs[1]) - P.qf_nreq) / P.qf_nreq;                                 // Eq. 70
  const double th_nu = atan2(raw[DP_NU_IM * M + i], raw[DP_NU_RE * M + i]);                                  // Eq. 69 (the fold factor 2 has no phase)
  const double th_b = atan2(raw[DP_BP_IM * M + i], raw[DP_BP_RE * M + i]);                                   // Eq. 68
  const double f = P.qf_beta * sin(th_nu - th_b);
  const cplx D = delta[i];
  delta[i] = make_double2(D.x + D.x * f - D.y * gt, D.y + D.y * f + D.x * gt);                               // Eq. 67
}
// out[i] (=, +=) Re t[i] for a field derivative
__global__ void k_real_acc(double* out, const cplx* t, int64_t M, int first) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < M) out[i] = (first ? 0.0 : out[i]) + t[i].x;
}
// one (folded) current component of each spin as a complex field pair, for the derivative engine
__global__ void k_j_to_cplx(const double* raw, int d, int sym, cplx* dst, int64_t M) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= M) return;
  const double a = raw[(DP_JA0 + d) * M + i], b = raw[(DP_JB0 + d) * M + i];
  dst[i] = make_double2(sym ? a + b : a, 0.0); dst[M + i] = make_double2(sym ? a + b : b, 0.0);
}
