/*
 * wslda_oracle.c -- CPU oracle (TEST INFRASTRUCTURE ONLY; see wslda_oracle.h).
 *
 * Follows arXiv 2602.08982 step by step, in the paper's order and notation.  No blocking, fusion or
 * reordering: every transform is a full round trip through a textbook radix-2 FFT, every density is a
 * loop over n in increasing order, every potential is evaluated pointwise from its formula.
 * OpenMP appears only as "parallel for" over independent spinors or lattice points.
 */
#include "wslda_oracle.h"
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;
#define PI 3.14159265358979323846264338327950288

struct orc_ctx {
  orc_params p;
  int nd, N[3], stride[3];
  int64_t M;
  double dV, Lperp;
  double* k[3];                         /* Eq. 25 wave numbers on each held axis */
  double *kperp2, *cpref;               /* per spinor: k_perp^2 and mult/L_perp (Eqs. 29, 30) */
  double *w_a, *w_b, mu_a, mu_b;
  double *rho_a, *rho_b, *tau_a, *tau_b, *ja, *jb;   /* raw (unfolded) sums; ja/jb are [3][M] */
  cplx   *nu;
  cplx   *bp;                           /* B' of Eq. 68, raw sum like nu */
  double *alpha_a, *alpha_b, *V_a, *V_b, *U_a, *U_b, *lap_a, *lap_b, *lambda, *geff, *vext_a, *vext_b;
  cplx   *delta, *dext;
  double *Aa, *Ab;                      /* current potentials A_sigma = dE/dj_sigma, [3][M] */
  double *vel_a, *vel_b;                /* external velocity fields v_ext_sigma, [3][M] */
  int lambda_valid;
};

/* ------------------------------------------------------------------------------------------------------ */
/* O1: transforms.  Forward: f~_l = sum_j f_j exp(-2 pi i j l / n) (Eq. 26 read with Eq. 25).               */

void orc_dft1d_naive(const double* in, double* out, int n, int sign) {
  for (int l = 0; l < n; ++l) {
    cplx s = 0.0;
    for (int j = 0; j < n; ++j) {
      double a = sign * 2.0 * PI * (double)(((int64_t)j * l) % n) / n;
      s += (in[2 * j] + I * in[2 * j + 1]) * (cos(a) + I * sin(a));
    }
    out[2 * l] = creal(s); out[2 * l + 1] = cimag(s);
  }
}

/* textbook iterative radix-2 decimation in time: bit-reversal permutation, then log2(n) butterfly levels;
 * every twiddle evaluated directly from cos/sin (no recurrence). */
int orc_fft1d(double* xr, int n, int sign) {
  if (n < 1 || (n & (n - 1))) return -1;
  cplx* x = (cplx*)xr;
  for (int i = 1, j = 0; i < n; ++i) {
    int bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) { cplx t = x[i]; x[i] = x[j]; x[j] = t; }
  }
  for (int len = 2; len <= n; len <<= 1) {
    int half = len >> 1;
    for (int s = 0; s < n; s += len)
      for (int q = 0; q < half; ++q) {
        double a = sign * 2.0 * PI * q / len;
        cplx w = cos(a) + I * sin(a);
        cplx u = x[s + q], v = w * x[s + q + half];
        x[s + q] = u + v; x[s + q + half] = u - v;
      }
  }
  return 0;
}

/* multi-dimensional transform over the held axes: 1-D transforms line by line, axis by axis */
static void fftnd(int nd, const int* N, cplx* a, int sign) {
  int64_t M = 1; for (int d = 0; d < nd; ++d) M *= N[d];
  for (int ax = 0; ax < nd; ++ax) {
    int64_t st = 1; for (int d = ax + 1; d < nd; ++d) st *= N[d];
    int n = N[ax];
    cplx* line = (cplx*)malloc(sizeof(cplx) * n);
    for (int64_t base = 0; base < M; ++base) {
      if ((base / st) % n) continue;            /* base runs over the points with index 0 on this axis */
      for (int j = 0; j < n; ++j) line[j] = a[base + j * st];
      orc_fft1d((double*)line, n, sign);
      for (int j = 0; j < n; ++j) a[base + j * st] = line[j];
    }
    free(line);
  }
}

static void make_k(int n, double dx, double* k) {   /* Eq. 25 */
  double L = n * dx;
  for (int l = 0; l < n; ++l) k[l] = (l < n / 2) ? 2.0 * PI * l / L : 2.0 * PI * (l - n) / L;
}

/* lap = sum_d d^2/dx_d^2 in (r = 2: all modes kept); grad_d = d/dx_d in (r = 1: Nyquist l = N_d/2 of that
 * axis set to zero).  Inverse transform carries 1/M. */
static void derivs(int nd, const int* N, double* const* k, const cplx* in, cplx* lap, cplx* grad) {
  int64_t M = 1; for (int d = 0; d < nd; ++d) M *= N[d];
  cplx* F = (cplx*)malloc(sizeof(cplx) * M);
  cplx* G = (cplx*)malloc(sizeof(cplx) * M);
  memcpy(F, in, sizeof(cplx) * M);
  fftnd(nd, N, F, -1);
  for (int which = -1; which < nd; ++which) {
    if (which < 0 && !lap) continue;
    if (which >= 0 && !grad) continue;
    for (int64_t i = 0; i < M; ++i) {
      int idx[3]; int64_t r = i;
      for (int d = nd - 1; d >= 0; --d) { idx[d] = (int)(r % N[d]); r /= N[d]; }
      if (which < 0) {
        double k2 = 0; for (int d = 0; d < nd; ++d) k2 += k[d][idx[d]] * k[d][idx[d]];
        G[i] = -k2 * F[i];
      } else {
        double kk = (idx[which] == N[which] / 2) ? 0.0 : k[which][idx[which]];
        G[i] = I * kk * F[i];
      }
    }
    fftnd(nd, N, G, +1);
    cplx* dst = (which < 0) ? lap : grad + (int64_t)which * M;
    for (int64_t i = 0; i < M; ++i) dst[i] = G[i] / (double)M;
  }
  free(F); free(G);
}

int orc_derivatives(int mode, const int dims[3], const double dx[3], const double* in, double* lap, double* grad) {
  if (mode < 1 || mode > 3) return -1;
  double* k[3] = {0, 0, 0};
  for (int d = 0; d < mode; ++d) {
    if (dims[d] < 2 || (dims[d] & (dims[d] - 1))) return -1;
    k[d] = (double*)malloc(sizeof(double) * dims[d]); make_k(dims[d], dx[d], k[d]);
  }
  derivs(mode, dims, k, (const cplx*)in, (cplx*)lap, (cplx*)grad);
  for (int d = 0; d < mode; ++d) free(k[d]);
  return 0;
}

/* ------------------------------------------------------------------------------------------------------ */
/* context                                                                                                  */

static double* dalloc(int64_t n) { return (double*)calloc((size_t)n, sizeof(double)); }

int orc_create(orc_ctx** out, const orc_params* p) {
  if (!out || !p || p->mode < 1 || p->mode > 3 || p->n_wf < 1) return -1;
  for (int d = 0; d < 3; ++d) if (p->dims[d] < 1 || p->dx[d] <= 0) return -1;
  for (int d = 0; d < p->mode; ++d) if (p->dims[d] < 2 || (p->dims[d] & (p->dims[d] - 1))) return -1;
  int ok = (p->ab_order == 3 && p->am_order == 4) || (p->ab_order == 4 && p->am_order == 4) ||
           (p->ab_order == 4 && p->am_order == 5) || (p->ab_order == 5 && p->am_order == 5);
  if (!ok || p->kin_form < 0 || p->kin_form > 2 || p->func_id < 0 || p->func_id > 2) return -1;
  orc_ctx* c = (orc_ctx*)calloc(1, sizeof(orc_ctx));
  c->p = *p; c->nd = p->mode; c->M = 1; c->dV = 1; c->Lperp = 1;
  for (int d = 0; d < 3; ++d) {
    if (d < c->nd) { c->N[d] = p->dims[d]; c->M *= p->dims[d]; c->dV *= p->dx[d]; }
    else c->Lperp *= p->dims[d] * p->dx[d];
  }
  for (int d = 0; d < c->nd; ++d) { c->k[d] = dalloc(c->N[d]); make_k(c->N[d], p->dx[d], c->k[d]); }
  int64_t M = c->M, n = p->n_wf;
  c->kperp2 = dalloc(n); c->cpref = dalloc(n); c->w_a = dalloc(n); c->w_b = dalloc(n);
  for (int64_t i = 0; i < n; ++i) { c->cpref[i] = 1.0 / c->Lperp; c->w_a[i] = 0.0; c->w_b[i] = 1.0; }
  c->rho_a = dalloc(M); c->rho_b = dalloc(M); c->tau_a = dalloc(M); c->tau_b = dalloc(M);
  c->ja = dalloc(3 * M); c->jb = dalloc(3 * M); c->nu = (cplx*)dalloc(2 * M); c->bp = (cplx*)dalloc(2 * M);
  c->alpha_a = dalloc(M); c->alpha_b = dalloc(M); c->V_a = dalloc(M); c->V_b = dalloc(M);
  c->U_a = dalloc(M); c->U_b = dalloc(M); c->lap_a = dalloc(M); c->lap_b = dalloc(M);
  c->lambda = dalloc(M); c->geff = dalloc(M); c->vext_a = dalloc(M); c->vext_b = dalloc(M);
  c->delta = (cplx*)dalloc(2 * M); c->dext = (cplx*)dalloc(2 * M);
  c->Aa = dalloc(3 * M); c->Ab = dalloc(3 * M); c->vel_a = dalloc(3 * M); c->vel_b = dalloc(3 * M);
  for (int64_t i = 0; i < M; ++i) c->alpha_a[i] = c->alpha_b[i] = 1.0;
  *out = c;
  return 0;
}

void orc_destroy(orc_ctx* c) {
  if (!c) return;
  double* v[] = {c->k[0], c->k[1], c->k[2], c->kperp2, c->cpref, c->w_a, c->w_b, c->rho_a, c->rho_b, c->tau_a,
                 c->tau_b, c->ja, c->jb, (double*)c->nu, c->alpha_a, c->alpha_b, c->V_a, c->V_b, c->U_a, c->U_b,
                 c->lap_a, c->lap_b, c->lambda, c->geff, c->vext_a, c->vext_b, (double*)c->delta, (double*)c->dext,
                 c->Aa, c->Ab, c->vel_a, c->vel_b, (double*)c->bp};
  for (size_t i = 0; i < sizeof(v) / sizeof(v[0]); ++i) free(v[i]);
  free(c);
}

int orc_set_modes(orc_ctx* c, int n_modes, const double* kperp, const double* mult, const int64_t* first) {
  if (!c || n_modes < 1 || first[0] != 0 || first[n_modes] != c->p.n_wf) return -1;
  for (int m = 0; m < n_modes; ++m) {
    if (first[m + 1] < first[m]) return -1;
    for (int64_t n = first[m]; n < first[m + 1]; ++n) {
      c->kperp2[n] = kperp[2 * m] * kperp[2 * m] + kperp[2 * m + 1] * kperp[2 * m + 1];
      c->cpref[n] = mult[m] / c->Lperp;
    }
  }
  return 0;
}

int orc_set_weights(orc_ctx* c, const double* w_a, const double* w_b) {
  memcpy(c->w_a, w_a, sizeof(double) * c->p.n_wf); memcpy(c->w_b, w_b, sizeof(double) * c->p.n_wf); return 0;
}
int orc_set_mu(orc_ctx* c, double mu_a, double mu_b) { c->mu_a = mu_a; c->mu_b = mu_b; return 0; }

int orc_set_external(orc_ctx* c, const double* va, const double* vb, const double* de) {
  int64_t M = c->M;
  if (va) memcpy(c->vext_a, va, sizeof(double) * M); else memset(c->vext_a, 0, sizeof(double) * M);
  if (vb) memcpy(c->vext_b, vb, sizeof(double) * M); else memset(c->vext_b, 0, sizeof(double) * M);
  if (de) memcpy(c->dext, de, sizeof(cplx) * M); else memset(c->dext, 0, sizeof(cplx) * M);
  return 0;
}

int orc_set_velocity(orc_ctx* c, const double* va, const double* vb) {
  int64_t M = c->M;
  if (va) memcpy(c->vel_a, va, sizeof(double) * 3 * M); else memset(c->vel_a, 0, sizeof(double) * 3 * M);
  if (vb) memcpy(c->vel_b, vb, sizeof(double) * 3 * M); else memset(c->vel_b, 0, sizeof(double) * 3 * M);
  return 0;
}

static void lap_of_real_field(orc_ctx* c, const double* f, double* lap) {
  int64_t M = c->M;
  cplx* a = (cplx*)malloc(sizeof(cplx) * M); cplx* l = (cplx*)malloc(sizeof(cplx) * M);
  for (int64_t i = 0; i < M; ++i) a[i] = f[i];
  derivs(c->nd, c->N, c->k, a, l, NULL);
  for (int64_t i = 0; i < M; ++i) lap[i] = creal(l[i]);
  free(a); free(l);
}

int orc_set_potentials(orc_ctx* c, const double* aa, const double* ab, const double* Ua, const double* Ub,
                       const double* delta) {
  int64_t M = c->M;
  memcpy(c->alpha_a, aa, sizeof(double) * M); memcpy(c->alpha_b, ab, sizeof(double) * M);
  memcpy(c->U_a, Ua, sizeof(double) * M); memcpy(c->U_b, Ub, sizeof(double) * M);
  memcpy(c->delta, delta, sizeof(cplx) * M);
  lap_of_real_field(c, c->alpha_a, c->lap_a); lap_of_real_field(c, c->alpha_b, c->lap_b);
  return 0;
}

/* densities as the functional sees them: raw sums, folded per Eq. 8 when spin_symmetric */
static void folded(const orc_ctx* c, int64_t i, double* ra, double* rb, double* ta, double* tb, cplx* nu,
                   double ja[3], double jb[3]) {
  if (c->p.spin_symmetric) {
    *ra = *rb = c->rho_a[i] + c->rho_b[i]; *ta = *tb = c->tau_a[i] + c->tau_b[i]; *nu = 2.0 * c->nu[i];
    for (int d = 0; d < 3; ++d) ja[d] = jb[d] = c->ja[d * c->M + i] + c->jb[d * c->M + i];
  } else {
    *ra = c->rho_a[i]; *rb = c->rho_b[i]; *ta = c->tau_a[i]; *tb = c->tau_b[i]; *nu = c->nu[i];
    for (int d = 0; d < 3; ++d) { ja[d] = c->ja[d * c->M + i]; jb[d] = c->jb[d * c->M + i]; }
  }
}

int orc_get_field(orc_ctx* c, int id, double* dst) {
  int64_t M = c->M;
  const double* src = NULL;
  switch (id) {
    case ORC_ALPHA_A: src = c->alpha_a; break; case ORC_ALPHA_B: src = c->alpha_b; break;
    case ORC_U_A: src = c->U_a; break; case ORC_U_B: src = c->U_b; break;
    case ORC_LAP_ALPHA_A: src = c->lap_a; break; case ORC_LAP_ALPHA_B: src = c->lap_b; break;
    case ORC_LAMBDA_C: src = c->lambda; break; case ORC_G_EFF: src = c->geff; break;
    case ORC_V_A: src = c->V_a; break; case ORC_V_B: src = c->V_b; break;
    case ORC_DELTA: memcpy(dst, c->delta, sizeof(cplx) * M); return 0;
    case ORC_BP:
      for (int64_t i = 0; i < M; ++i) { cplx b = (c->p.spin_symmetric ? 2.0 : 1.0) * c->bp[i]; dst[2 * i] = creal(b); dst[2 * i + 1] = cimag(b); }
      return 0;
    default: break;
  }
  if (id >= ORC_AA_X && id <= ORC_AB_Z) src = (id <= ORC_AA_Z ? c->Aa + (id - ORC_AA_X) * M : c->Ab + (id - ORC_AB_X) * M);
  if (src) { memcpy(dst, src, sizeof(double) * M); return 0; }
  if (id < 0 || id > ORC_JB_Z) return -1;
  for (int64_t i = 0; i < M; ++i) {
    double ra, rb, ta, tb, ja[3], jb[3]; cplx nu;
    folded(c, i, &ra, &rb, &ta, &tb, &nu, ja, jb);
    switch (id) {
      case ORC_RHO_A: dst[i] = ra; break; case ORC_RHO_B: dst[i] = rb; break;
      case ORC_TAU_A: dst[i] = ta; break; case ORC_TAU_B: dst[i] = tb; break;
      case ORC_NU: dst[2 * i] = creal(nu); dst[2 * i + 1] = cimag(nu); break;
      default: dst[i] = (id <= ORC_JA_Z) ? ja[id - ORC_JA_X] : jb[id - ORC_JB_X];
    }
  }
  return 0;
}

int orc_set_field(orc_ctx* c, int id, const double* src) {
  int64_t M = c->M;
  switch (id) {
    case ORC_RHO_A: memcpy(c->rho_a, src, 8 * M); return 0; case ORC_RHO_B: memcpy(c->rho_b, src, 8 * M); return 0;
    case ORC_TAU_A: memcpy(c->tau_a, src, 8 * M); return 0; case ORC_TAU_B: memcpy(c->tau_b, src, 8 * M); return 0;
    case ORC_NU: memcpy(c->nu, src, 16 * M); return 0;
    case ORC_LAMBDA_C: memcpy(c->lambda, src, 8 * M); c->lambda_valid = 1; return 0;
    default: return -1;
  }
}

/* ------------------------------------------------------------------------------------------------------ */
/* O2: H psi for one spinor (Eqs. 5, 15; h from Eq. 4c without the anticommutator term; kinetic operator
 * Eq. 14 / Eq. 40 / successive first derivatives; transverse substitution mu -> mu - alpha k_perp^2/2,
 * PAPER.md:413-419, 444-448).                                                                              */

static void kinetic(const orc_ctx* c, const cplx* w, const double* alpha, const double* lap_alpha, double kp2, cplx* out) {
  int64_t M = c->M; int nd = c->nd;
  cplx* lap = (cplx*)malloc(sizeof(cplx) * M);
  if (c->p.kin_form == 0) {                                   /* Eq. 14: K w = -1/2 lap w + 1/2 k_perp^2 w */
    derivs(nd, c->N, c->k, w, lap, NULL);
    for (int64_t i = 0; i < M; ++i) out[i] = -0.5 * lap[i] + 0.5 * kp2 * w[i];
  } else if (c->p.kin_form == 1) {                            /* Eq. 40 summed over the held axes */
    cplx* aw = (cplx*)malloc(sizeof(cplx) * M); cplx* lap_aw = (cplx*)malloc(sizeof(cplx) * M);
    for (int64_t i = 0; i < M; ++i) aw[i] = alpha[i] * w[i];
    derivs(nd, c->N, c->k, w, lap, NULL);
    derivs(nd, c->N, c->k, aw, lap_aw, NULL);
    for (int64_t i = 0; i < M; ++i)
      out[i] = -0.25 * (lap_aw[i] + alpha[i] * lap[i] - lap_alpha[i] * w[i]) + 0.5 * alpha[i] * kp2 * w[i];
    free(aw); free(lap_aw);
  } else {                                                    /* -1/2 sum_j d_j (alpha d_j w) */
    cplx* g = (cplx*)malloc(sizeof(cplx) * M * nd); cplx* g2 = (cplx*)malloc(sizeof(cplx) * M * nd);
    derivs(nd, c->N, c->k, w, NULL, g);
    for (int64_t i = 0; i < M; ++i) out[i] = 0.5 * alpha[i] * kp2 * w[i];
    for (int d = 0; d < nd; ++d) {
      for (int64_t i = 0; i < M; ++i) g[d * M + i] *= alpha[i];
      derivs(nd, c->N, c->k, g + d * M, NULL, g2);
      for (int64_t i = 0; i < M; ++i) out[i] += -0.5 * g2[d * M + i];
    }
    free(g); free(g2);
  }
  free(lap);
}

/* The current / velocity coupling of Eq. 4c: out += -(i/2) {W, grad} w with W = A_sigma - v_ext_sigma real,
 * {W, grad} w = W . grad w + grad . (W w) over the held axes, both derivatives spectral with the Nyquist rule of an odd
 * derivative.  In this form the discrete operator is exactly Hermitian (R27). */
static void add_current_term(const orc_ctx* c, const cplx* w, const double* A, const double* vel, cplx* out) {
  int64_t M = c->M; int nd = c->nd;
  cplx* g = (cplx*)malloc(sizeof(cplx) * M * nd); cplx* Ww = (cplx*)malloc(sizeof(cplx) * M);
  cplx* g2 = (cplx*)malloc(sizeof(cplx) * M * nd);
  derivs(nd, c->N, c->k, w, NULL, g);
  for (int d = 0; d < nd; ++d) {
    for (int64_t i = 0; i < M; ++i) Ww[i] = (A[d * M + i] - vel[d * M + i]) * w[i];
    derivs(nd, c->N, c->k, Ww, NULL, g2);
    for (int64_t i = 0; i < M; ++i)
      out[i] += -0.5 * I * ((A[d * M + i] - vel[d * M + i]) * g[d * M + i] + g2[d * M + i]);
  }
  free(g); free(Ww); free(g2);
}

static double apply_h_one(const orc_ctx* c, int64_t n, const cplx* psi, cplx* hpsi) {
  int64_t M = c->M;
  const cplx *u = psi, *v = psi + M;
  cplx* Ku = (cplx*)malloc(sizeof(cplx) * M); cplx* Kv = (cplx*)malloc(sizeof(cplx) * M);
  kinetic(c, u, c->alpha_a, c->lap_a, c->kperp2[n], Ku);
  kinetic(c, v, c->alpha_b, c->lap_b, c->kperp2[n], Kv);
  if (c->p.current_terms) {
    /* row u: h_a u.  Row v: -h_b^* v, and the conjugate of -(i/2){W, grad} is +(i/2){W, grad}, so that
     * -h_b^* v = -(K_b + U_b) v - (i/2){W_b, grad} v: the coupling enters Kv with the opposite sign (Eq. 4b) */
    add_current_term(c, u, c->Aa, c->vel_a, Ku);
    for (int64_t i = 0; i < M; ++i) Kv[i] = -Kv[i];
    add_current_term(c, v, c->Ab, c->vel_b, Kv);
    for (int64_t i = 0; i < M; ++i) Kv[i] = -Kv[i];
  }
  cplx e = 0.0;
  for (int64_t i = 0; i < M; ++i) {
    cplx D = c->delta[i] + c->dext[i];
    cplx hu = Ku[i] + (c->U_a[i] - c->mu_a) * u[i] + D * v[i];
    cplx hv = conj(D) * u[i] - (Kv[i] + (c->U_b[i] - c->mu_b) * v[i]);
    hpsi[i] = hu; hpsi[M + i] = hv;
    e += conj(u[i]) * hu + conj(v[i]) * hv;                 /* Eq. 44b */
  }
  free(Ku); free(Kv);
  return creal(e) * c->dV;
}

int orc_apply_h(orc_ctx* c, const double* psi, double* hpsi, double* eps, int64_t n_first, int64_t n_count) {
  if (!c || n_first < 0 || n_first + n_count > c->p.n_wf) return -1;
  int64_t M = c->M;
#pragma omp parallel for schedule(static)
  for (int64_t n = n_first; n < n_first + n_count; ++n) {
    double e = apply_h_one(c, n, (const cplx*)psi + 2 * M * n, (cplx*)hpsi + 2 * M * n);
    if (eps) eps[n] = e;
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------------------ */
/* O4: densities, Eqs. 7a-g; prefactors and k_perp terms of Eqs. 29b-e / 30b-e.         */

int orc_densities(orc_ctx* c, const double* psi_, int64_t n_first, int64_t n_count, int accumulate) {
  if (!c || n_first < 0 || n_first + n_count > c->p.n_wf) return -1;
  int64_t M = c->M; int nd = c->nd;
  const cplx* psi = (const cplx*)psi_;
  if (!accumulate) {
    memset(c->rho_a, 0, 8 * M); memset(c->rho_b, 0, 8 * M); memset(c->tau_a, 0, 8 * M); memset(c->tau_b, 0, 8 * M);
    memset(c->ja, 0, 24 * M); memset(c->jb, 0, 24 * M); memset(c->nu, 0, 16 * M); memset(c->bp, 0, 16 * M);
  }
  const int64_t CH = 64;                       /* gradients of CH spinors at a time, then sum them in n order */
  cplx* g = (cplx*)malloc(sizeof(cplx) * CH * 2 * nd * M);
  cplx* lp = (cplx*)malloc(sizeof(cplx) * CH * 2 * M);          /* Laplacians, for B' of Eq. 68 */
  for (int64_t n0 = n_first; n0 < n_first + n_count; n0 += CH) {
    int64_t nc = (n_first + n_count - n0 < CH) ? n_first + n_count - n0 : CH;
#pragma omp parallel for schedule(static)
    for (int64_t q = 0; q < 2 * nc; ++q) {
      int64_t n = n0 + q / 2; int comp = (int)(q % 2);
      derivs(nd, c->N, c->k, psi + (2 * n + comp) * M, lp + q * M, g + q * nd * M);
    }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < M; ++i)
      for (int64_t s = 0; s < nc; ++s) {
        int64_t n = n0 + s;
        cplx u = psi[2 * n * M + i], v = psi[(2 * n + 1) * M + i];
        double cw_a = c->cpref[n] * c->w_a[n], cw_b = c->cpref[n] * c->w_b[n];
        const cplx* gu = g + (2 * s) * nd * M; const cplx* gv = g + (2 * s + 1) * nd * M;
        double u2 = creal(u) * creal(u) + cimag(u) * cimag(u), v2 = creal(v) * creal(v) + cimag(v) * cimag(v);
        double gu2 = 0, gv2 = 0;
        for (int d = 0; d < nd; ++d) {
          cplx a = gu[d * M + i], b = gv[d * M + i];
          gu2 += creal(a) * creal(a) + cimag(a) * cimag(a); gv2 += creal(b) * creal(b) + cimag(b) * cimag(b);
          c->ja[d * M + i] += -cw_a * cimag(u * conj(a));                  /* Eq. 7f */
          c->jb[d * M + i] += cw_b * cimag(v * conj(b));                   /* Eq. 7g */
        }
        {                                                                    /* Eq. 68 (reading R29): the weights of nu; the
                                                                                plane-wave factor turns lap into lap - k_perp^2 */
          cplx lu = lp[(2 * s) * M + i] - c->kperp2[n] * u, lv = lp[(2 * s + 1) * M + i] - c->kperp2[n] * v;
          c->bp[i] += -0.5 * 0.5 * c->cpref[n] * (c->w_b[n] - c->w_a[n]) * (u * conj(lv) + conj(v) * lu);
        }
        c->rho_a[i] += cw_a * u2;                                            /* Eq. 7a */
        c->rho_b[i] += cw_b * v2;                                            /* Eq. 7b */
        c->tau_a[i] += cw_a * (gu2 + c->kperp2[n] * u2);                     /* Eq. 7c, 29c, 30c */
        c->tau_b[i] += cw_b * (gv2 + c->kperp2[n] * v2);                     /* Eq. 7d */
        c->nu[i] += 0.5 * c->cpref[n] * (c->w_b[n] - c->w_a[n]) * u * conj(v);   /* Eq. 7e */
      }
  }
  free(g); free(lp);
  return 0;
}

/* ------------------------------------------------------------------------------------------------------ */
/* O5: pointwise functional.  Eqs. 9c-d, 10, 11, 12a-c, 19-22; V_sigma = dE/d rho_sigma.     */

static double A_of(double p) { return 1.094 + 0.156 * p * (1 - 2 * p * p / 3 + p * p * p * p / 5) - 0.532 * p * p * (1 - p * p + p * p * p * p / 3); }
static double dA_of(double p) { double q = 1 - p * p; return q * q * (0.156 - 1.064 * p); }

static double lambda_c(double alpha_p, double V_p, double mu_p, double E_c, int* window_empty) {
  double k02 = 2.0 * (mu_p - V_p) / alpha_p;            /* Eq. 21a */
  double kc2 = 2.0 * (E_c + mu_p - V_p) / alpha_p;      /* Eq. 21b */
  *window_empty = 0;
  if (kc2 <= 0) { *window_empty = 1; return 0.0; }
  double kc = sqrt(kc2);
  if (k02 > 0) {                                         /* Eq. 20 */
    double k0 = sqrt(k02);
    return kc / (2 * PI * PI * alpha_p) * (1.0 - k0 / (2 * kc) * log((kc + k0) / (kc - k0)));
  }
  /* k0^2 <= 0 (outside the cloud): Eq. 20 is the closed form of (1/2 pi^2 alpha) PV int_0^kc k^2 dk/(k^2-k0^2);
   * for k0^2 = -kap^2 the same integral is regular and equals kc - kap atan(kc/kap)  (R5) */
  double kap = sqrt(-k02);
  if (kap == 0.0) return kc / (2 * PI * PI * alpha_p);
  return kc / (2 * PI * PI * alpha_p) * (1.0 - kap / kc * atan(kc / kap));
}

int orc_functional_point(const orc_ctx* c, const double in[9], int use_lambda_in, double out[10]) {
  const double z[3] = {0, 0, 0}; double A[6];
  return orc_functional_point_j(c, in, z, z, use_lambda_in, out, A);
}

int orc_functional_point_j(const orc_ctx* c, const double in[9], const double ja[3], const double jb[3], int use_lambda_in,
                           double out[10], double A_out[6]) {
  double ra = in[0], rb = in[1], ta = in[2], tb = in[3]; cplx nu = in[4] + I * in[5];
  double ja2 = ja[0] * ja[0] + ja[1] * ja[1] + ja[2] * ja[2], jb2 = jb[0] * jb[0] + jb[1] * jb[1] + jb[2] * jb[2];
  for (int d = 0; d < 6; ++d) A_out[d] = 0;
  double va = in[6], vb = in[7];
  double rho = ra + rb; if (rho < c->p.rho_floor) rho = c->p.rho_floor;
  double aa = 1, ab = 1, Va0 = 0, Vb0 = 0, edens = 0, inv_g0;
  if (c->p.func_id == 1) {                               /* BdG: A=1, B=0, C/rho^(1/3) = 4 pi a_s */
    inv_g0 = 1.0 / c->p.four_pi_as;
    edens = 0.5 * ta + 0.5 * tb;
  } else {
    double p = (ra - rb) / rho; if (p > 1) p = 1; if (p < -1) p = -1;
    double dAp = 0, dAm = 0;
    if (!c->p.force_a1) { aa = A_of(p); ab = A_of(-p); dAp = dA_of(p); dAm = dA_of(-p); }
    double sp = 0.5 * (1 + p), sm = 0.5 * (1 - p), c23 = cbrt(4.0);
    double B = c23 * (0.357 + 0.642 * p * p - aa * pow(sp, 5.0 / 3) - ab * pow(sm, 5.0 / 3));       /* Eq. 12b */
    double dB = c23 * (1.284 * p - dAp * pow(sp, 5.0 / 3) - (5.0 / 6) * aa * pow(sp, 2.0 / 3)
                                 + dAm * pow(sm, 5.0 / 3) + (5.0 / 6) * ab * pow(sm, 2.0 / 3));
    double eF = 0.5 * pow(3 * PI * PI * rho, 2.0 / 3);                                              /* Eq. 9d */
    double dp_a = 2 * rb / (rho * rho), dp_b = -2 * ra / (rho * rho);
    double common = 0.5 * dAp * ta - 0.5 * dAm * tb + 0.6 * rho * eF * dB;
    Va0 = common * dp_a + B * eF;
    Vb0 = common * dp_b + B * eF;
    inv_g0 = cbrt(rho) / c->p.C;
    edens = 0.5 * aa * ta + 0.5 * ab * tb + 0.6 * B * rho * eF;
    if (c->p.current_terms) {
      /* E_CM + the j-part of E_0 (Eqs. 9b, 9c): sum_sigma (1 - alpha_sigma) j_sigma^2 / (2 rho_sigma);
       * A_sigma = dE/dj_sigma; V_sigma += dE/drho_sigma of that term, alpha_a = A(p), alpha_b = A(-p) */
      double rsa = ra < c->p.rho_floor ? c->p.rho_floor : ra, rsb = rb < c->p.rho_floor ? c->p.rho_floor : rb;
      edens += 0.5 * (1 - aa) * ja2 / rsa + 0.5 * (1 - ab) * jb2 / rsb;
      for (int d = 0; d < 3; ++d) { A_out[d] = (1 - aa) * ja[d] / rsa; A_out[3 + d] = (1 - ab) * jb[d] / rsb; }
      double dal = -0.5 * dAp * ja2 / rsa + 0.5 * dAm * jb2 / rsb;      /* through d alpha_sigma / dp */
      Va0 += dal * dp_a - 0.5 * (1 - aa) * ja2 / (rsa * rsa);
      Vb0 += dal * dp_b - 0.5 * (1 - ab) * jb2 / (rsb * rsb);
    }
  }
  int empty = 0;
  double lam = use_lambda_in ? in[8]
             : lambda_c(0.5 * (aa + ab), 0.5 * (Va0 + va + Vb0 + vb), 0.5 * (c->mu_a + c->mu_b), c->p.E_cut, &empty);
  double g = empty ? 0.0 : 1.0 / (inv_g0 - lam);         /* Eq. 19 in the reading of DESIGN.md R1 */
  cplx D = -g * nu;                                       /* Eq. 10 */
  double D2 = creal(D) * creal(D) + cimag(D) * cimag(D);
  double Va = Va0, Vb = Vb0;
  if (c->p.func_id == 2) { double t = D2 / (3.0 * c->p.C * pow(rho, 2.0 / 3)); Va -= t; Vb -= t; }
  edens += g * (creal(nu) * creal(nu) + cimag(nu) * cimag(nu));
  out[0] = aa; out[1] = ab; out[2] = Va; out[3] = Vb; out[4] = creal(D); out[5] = cimag(D);
  out[6] = lam; out[7] = g; out[8] = edens; out[9] = 0;
  return 0;
}

int orc_update_potentials(orc_ctx* c) {
  if (c->p.func_id == 0) return 0;                       /* fixed potentials: nothing to rebuild */
  int64_t M = c->M;
  int frozen = c->p.lambda_mode == 1 && c->lambda_valid;
  for (int64_t i = 0; i < M; ++i) {
    double ra, rb, ta, tb, ja[3], jb[3], in[9], out[10], A[6]; cplx nu;
    folded(c, i, &ra, &rb, &ta, &tb, &nu, ja, jb);
    in[0] = ra; in[1] = rb; in[2] = ta; in[3] = tb; in[4] = creal(nu); in[5] = cimag(nu);
    in[6] = c->vext_a[i]; in[7] = c->vext_b[i]; in[8] = c->lambda[i];
    orc_functional_point_j(c, in, ja, jb, frozen, out, A);
    for (int d = 0; d < 3; ++d) { c->Aa[d * M + i] = A[d]; c->Ab[d * M + i] = A[3 + d]; }
    c->alpha_a[i] = out[0]; c->alpha_b[i] = out[1]; c->V_a[i] = out[2]; c->V_b[i] = out[3];
    c->delta[i] = out[4] + I * out[5]; c->lambda[i] = out[6]; c->geff[i] = out[7];
    c->U_a[i] = c->V_a[i] + c->vext_a[i]; c->U_b[i] = c->V_b[i] + c->vext_b[i];
  }
  c->lambda_valid = 1;
  lap_of_real_field(c, c->alpha_a, c->lap_a); lap_of_real_field(c, c->alpha_b, c->lap_b);
  if (c->p.quantum_friction) {
    /* Eqs. 66-70: V_sigma += -(alpha_qf / rho_0) div j_sigma;
     * Delta += Delta [beta_qf sin(theta_nu - theta_B') + i gamma_qf (N - N_req) / N_req] */
    int nd = c->nd;
    cplx* f = (cplx*)malloc(sizeof(cplx) * M); cplx* gr = (cplx*)malloc(sizeof(cplx) * M * nd);
    double* dv[2] = {dalloc(M), dalloc(M)};
    double N = 0;
    for (int64_t i = 0; i < M; ++i) {
      double ra, rb, ta, tb, ja[3], jb[3]; cplx nu;
      folded(c, i, &ra, &rb, &ta, &tb, &nu, ja, jb);
      N += (ra + rb) * c->dV * c->Lperp;
    }
    for (int sg = 0; sg < 2; ++sg)
      for (int d = 0; d < nd; ++d) {
        for (int64_t i = 0; i < M; ++i) {
          double ra, rb, ta, tb, ja[3], jb[3]; cplx nu;
          folded(c, i, &ra, &rb, &ta, &tb, &nu, ja, jb);
          f[i] = sg ? jb[d] : ja[d];
        }
        derivs(nd, c->N, c->k, f, NULL, gr);
        for (int64_t i = 0; i < M; ++i) dv[sg][i] += creal(gr[d * M + i]);
      }
    double gt = c->p.qf_gamma * (N - c->p.qf_nreq) / c->p.qf_nreq;                        /* Eq. 70 */
    for (int64_t i = 0; i < M; ++i) {
      double Vd_a = -c->p.qf_alpha / c->p.qf_rho0 * dv[0][i], Vd_b = -c->p.qf_alpha / c->p.qf_rho0 * dv[1][i];   /* Eq. 66 */
      c->V_a[i] += Vd_a; c->V_b[i] += Vd_b; c->U_a[i] += Vd_a; c->U_b[i] += Vd_b;
      double f2 = c->p.spin_symmetric ? 2.0 : 1.0;
      cplx nu = f2 * c->nu[i], bp = f2 * c->bp[i];
      double th_nu = atan2(cimag(nu), creal(nu)), th_b = atan2(cimag(bp), creal(bp));      /* Eqs. 69, 68 */
      c->delta[i] += c->delta[i] * (c->p.qf_beta * sin(th_nu - th_b) + I * gt);           /* Eq. 67 */
    }
    free(f); free(gr); free(dv[0]); free(dv[1]);
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------------------ */
/* O3, O6, O7: right-hand side, ABM step (Alg. 2), Taylor starter                                          */

static const double AB3[3] = {23.0 / 12, -16.0 / 12, 5.0 / 12};                                   /* Eq. 46 */
static const double AB4[4] = {55.0 / 24, -59.0 / 24, 37.0 / 24, -9.0 / 24};                       /* Eq. 47 */
static const double AB5[5] = {1901.0 / 720, -2774.0 / 720, 2616.0 / 720, -1274.0 / 720, 251.0 / 720}; /* Eq. 48 */
static const double AM4[4] = {9.0 / 24, 19.0 / 24, -5.0 / 24, 1.0 / 24};                          /* Eq. 49 */
static const double AM5[5] = {251.0 / 720, 646.0 / 720, -264.0 / 720, 106.0 / 720, -19.0 / 720};  /* Eq. 50 */

int orc_history_length(const orc_ctx* c) { return c->p.ab_order > c->p.am_order - 1 ? c->p.ab_order : c->p.am_order - 1; }
int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

static void normalise(const orc_ctx* c, cplx* psi) {      /* Eq. 16 with n = m; Alg. 2 steps 2, 8 */
  int64_t M = c->M;
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < c->p.n_wf; ++n) {
    cplx* s = psi + 2 * M * n; double a = 0;
    for (int64_t i = 0; i < 2 * M; ++i) a += creal(s[i]) * creal(s[i]) + cimag(s[i]) * cimag(s[i]);
    double f = 1.0 / sqrt(a * c->dV);
    for (int64_t i = 0; i < 2 * M; ++i) s[i] *= f;
  }
}

static void rebuild(orc_ctx* c, const cplx* psi) {
  if (c->p.func_id == 0) return;
  orc_densities(c, (const double*)psi, 0, c->p.n_wf, 0);
  orc_update_potentials(c);
}

/* f(psi) = -i [H(psi) - <H>_n] psi, Eq. 45b; the potentials in H are those of psi itself */
static void rhs(orc_ctx* c, const cplx* psi, cplx* f) {
  int64_t M = c->M, n_wf = c->p.n_wf;
  rebuild(c, psi);
  double* eps = dalloc(n_wf);
  orc_apply_h(c, (const double*)psi, (double*)f, eps, 0, n_wf);
#pragma omp parallel for schedule(static)
  for (int64_t n = 0; n < n_wf; ++n) {
    double e = c->p.subtract_mean_energy ? eps[n] : 0.0;
    for (int64_t i = 2 * M * n; i < 2 * M * (n + 1); ++i) f[i] = -I * (f[i] - e * psi[i]);
  }
  free(eps);
}

/* Eqs. 53/54: out = sum_{k<=r} (-i s)^k / k! G^k phi with G = H - <H>_n (current potentials, eps fixed) */
static void taylor(orc_ctx* c, const cplx* phi, double s, int r, cplx* out) {
  int64_t M = c->M, n_wf = c->p.n_wf, tot = 2 * M * n_wf;
  cplx* t = (cplx*)malloc(sizeof(cplx) * tot); cplx* ht = (cplx*)malloc(sizeof(cplx) * tot);
  double* eps = dalloc(n_wf); double* dummy = dalloc(n_wf);
  memcpy(t, phi, sizeof(cplx) * tot); memcpy(out, phi, sizeof(cplx) * tot);
  cplx coef = 1.0;
  for (int k = 1; k <= r; ++k) {
    orc_apply_h(c, (const double*)t, (double*)ht, k == 1 ? eps : dummy, 0, n_wf);
    if (k == 1 && !c->p.subtract_mean_energy) memset(eps, 0, sizeof(double) * n_wf);
    coef *= (-I * s) / (double)k;
#pragma omp parallel for schedule(static)
    for (int64_t n = 0; n < n_wf; ++n)
      for (int64_t i = 2 * M * n; i < 2 * M * (n + 1); ++i) {
        cplx g = ht[i] - eps[n] * t[i];
        t[i] = g; out[i] += coef * g;
      }
  }
  free(t); free(ht); free(eps); free(dummy);
}

static void rotate_history(double** f_hist, int m) {     /* Alg. 2 steps 5-7: f_i -> f_{i+1}; oldest buffer becomes slot 0 */
  double* last = f_hist[m - 1];
  for (int i = m - 1; i > 0; --i) f_hist[i] = f_hist[i - 1];
  f_hist[0] = last;
}

int orc_abm_init(orc_ctx* c, double* phi_, double** f_hist, double dt, int selfstart) {
  int m = orc_history_length(c);
  int64_t tot = 2 * c->M * c->p.n_wf;
  cplx* phi = (cplx*)phi_;
  if (!selfstart) {                                      /* stationary start: f_k = 0 by definition */
    for (int i = 0; i < m; ++i) memset(f_hist[i], 0, sizeof(cplx) * tot);
    rebuild(c, phi);
    return 0;
  }
  int r = c->p.am_order;                                 /* truncation order = corrector order */
  cplx* pred = (cplx*)malloc(sizeof(cplx) * tot); cplx* next = (cplx*)malloc(sizeof(cplx) * tot);
  rhs(c, phi, (cplx*)f_hist[0]);
  for (int s = 1; s < m; ++s) {
    taylor(c, phi, 0.5 * dt, r, pred);                   /* Eq. 53 */
    rebuild(c, pred);                                    /* H(phi^(p), t + dt/2) */
    taylor(c, phi, dt, r, next);                         /* Eq. 54 */
    if (c->p.normalize) normalise(c, next);
    memcpy(phi, next, sizeof(cplx) * tot);
    rotate_history(f_hist, m);
    rhs(c, phi, (cplx*)f_hist[0]);
  }
  free(pred); free(next);
  return 0;
}

int orc_abm_step(orc_ctx* c, double* phi_, double** f_hist, double dt) {
  int m = orc_history_length(c), ab = c->p.ab_order, am = c->p.am_order;
  const double* b = ab == 3 ? AB3 : ab == 4 ? AB4 : AB5;
  const double* cc = am == 4 ? AM4 : AM5;
  int64_t tot = 2 * c->M * c->p.n_wf;
  cplx* phi = (cplx*)phi_;
  cplx* P = (cplx*)malloc(sizeof(cplx) * tot); cplx* Cp = (cplx*)malloc(sizeof(cplx) * tot);
  cplx* g = (cplx*)malloc(sizeof(cplx) * tot);
  /* step 1: predictor (Eqs. 46-48) and the known part of the corrector (Eqs. 49-50), simultaneously */
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < tot; ++i) {
    cplx p = phi[i], q = phi[i];
    for (int j = 0; j < ab; ++j) p += b[j] * dt * ((const cplx*)f_hist[j])[i];
    for (int j = 1; j < am; ++j) q += cc[j] * dt * ((const cplx*)f_hist[j - 1])[i];
    P[i] = p; Cp[i] = q;
  }
  if (c->p.normalize) normalise(c, P);                   /* step 2 */
  rhs(c, P, g);                                          /* step 3 */
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < tot; ++i) phi[i] = Cp[i] + cc[0] * dt * g[i];   /* step 4 */
  rotate_history(f_hist, m);                             /* steps 5-7 */
  if (c->p.normalize) normalise(c, phi);                 /* step 8 */
  rhs(c, phi, (cplx*)f_hist[0]);                         /* step 9 */
  free(P); free(Cp); free(g);
  return 0;
}

/* O8: Eqs. 33a-g with the in-scope energy density (no current terms) */
int orc_energy(orc_ctx* c, double out[10]) {
  int64_t M = c->M; double dVf = c->dV * c->Lperp;
  for (int q = 0; q < 10; ++q) out[q] = 0;
  for (int64_t i = 0; i < M; ++i) {
    double ra, rb, ta, tb, ja[3], jb[3]; cplx nu;
    folded(c, i, &ra, &rb, &ta, &tb, &nu, ja, jb);
    out[0] += ra * dVf; out[1] += rb * dVf;
    out[2] += 0.5 * (c->alpha_a[i] * ta + c->alpha_b[i] * tb) * dVf;                        /* 33a */
    if (c->p.current_terms) {
      double rsa = ra < c->p.rho_floor ? c->p.rho_floor : ra, rsb = rb < c->p.rho_floor ? c->p.rho_floor : rb;
      double ja2 = ja[0] * ja[0] + ja[1] * ja[1] + ja[2] * ja[2], jb2 = jb[0] * jb[0] + jb[1] * jb[1] + jb[2] * jb[2];
      out[2] -= 0.5 * (c->alpha_a[i] * ja2 / rsa + c->alpha_b[i] * jb2 / rsb) * dVf;         /* 33a, the -j^2/rho part */
      out[8] += 0.5 * (ja2 / rsa + jb2 / rsb) * dVf;                                         /* 33d */
      for (int d = 0; d < 3; ++d) out[9] -= (c->vel_a[d * M + i] * ja[d] + c->vel_b[d * M + i] * jb[d]) * dVf;   /* 33g */
    }
    if (c->p.func_id == 2) {
      double rho = ra + rb; if (rho < c->p.rho_floor) rho = c->p.rho_floor;
      double p = (ra - rb) / rho; if (p > 1) p = 1; if (p < -1) p = -1;
      double B = cbrt(4.0) * (0.357 + 0.642 * p * p - c->alpha_a[i] * pow(0.5 * (1 + p), 5.0 / 3) - c->alpha_b[i] * pow(0.5 * (1 - p), 5.0 / 3));
      out[3] += 0.6 * B * rho * 0.5 * pow(3 * PI * PI * rho, 2.0 / 3) * dVf;                /* 33b */
    }
    out[4] += -creal(conj(c->delta[i]) * nu) * dVf;                                         /* 33c */
    out[5] += (c->vext_a[i] * ra + c->vext_b[i] * rb) * dVf;                                /* 33e */
    out[6] += -2.0 * creal(c->dext[i] * conj(nu)) * dVf;                                    /* 33f */
  }
  out[7] = out[2] + out[3] + out[4] + out[5] + out[6] + out[8] + out[9];
  return 0;
}
