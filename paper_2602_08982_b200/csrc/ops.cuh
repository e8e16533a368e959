// ops.cuh -- setters, the derivative engine dispatch, and the three single-call entry points
// wslda_apply_h / wslda_densities / wslda_update_potentials (general chunked path).
#pragma once
#include "ctx.cuh"

static inline cudaStream_t S(void* s) { return (cudaStream_t)s; }
static inline unsigned nb(int64_t n, int t) { return (unsigned)((n + t - 1) / t); }

extern "C" wslda_status wslda_set_modes(wslda_ctx* c, int n_modes, const double* kperp, const double* mult, const int64_t* first,
                                        void* stream) {
  if (!c) return WSLDA_EINVAL;
  if (n_modes < 1 || !kperp || !mult || !first || first[0] != 0 || first[n_modes] != c->P.n_wf)
    return fail(c, WSLDA_EINVAL, "set_modes: first[] must run from 0 to n_wf");
  const int64_t n_wf = c->P.n_wf;
  std::vector<double> k2(n_wf), cp(n_wf);
  for (int m = 0; m < n_modes; ++m) {
    if (first[m + 1] < first[m]) return fail(c, WSLDA_EINVAL, "set_modes: first[] must be non-decreasing");
    for (int64_t n = first[m]; n < first[m + 1]; ++n) {
      k2[n] = kperp[2 * m] * kperp[2 * m] + kperp[2 * m + 1] * kperp[2 * m + 1];
      cp[n] = mult[m] / c->Lperp;
    }
  }
  // pageable host source: the runtime stages the data before returning, the device copy is ordered on the stream
  cudaMemcpyAsync(c->kperp2, k2.data(), n_wf * 8, cudaMemcpyHostToDevice, S(stream));
  cudaMemcpyAsync(c->cpref, cp.data(), n_wf * 8, cudaMemcpyHostToDevice, S(stream));
  return cuda_check(c, "set_modes");
}

extern "C" wslda_status wslda_set_weights(wslda_ctx* c, const double* w_a, const double* w_b, void* stream) {
  if (!c || !w_a || !w_b) return fail(c, WSLDA_EINVAL, "set_weights: null argument");
  cudaMemcpyAsync(c->w_a, w_a, c->P.n_wf * 8, cudaMemcpyDeviceToDevice, S(stream));
  cudaMemcpyAsync(c->w_b, w_b, c->P.n_wf * 8, cudaMemcpyDeviceToDevice, S(stream));
  return cuda_check(c, "set_weights");
}

extern "C" wslda_status wslda_set_mu(wslda_ctx* c, double mu_a, double mu_b) {
  if (!c) return WSLDA_EINVAL;
  c->mu_a = mu_a; c->mu_b = mu_b;
  return WSLDA_OK;
}

extern "C" wslda_status wslda_set_external(wslda_ctx* c, const double* va, const double* vb, const void* de, void* stream) {
  if (!c) return WSLDA_EINVAL;
  const int64_t M = c->P.M;
  cudaStream_t st = S(stream);
  if (va) cudaMemcpyAsync(c->vext_a, va, M * 8, cudaMemcpyDeviceToDevice, st); else cudaMemsetAsync(c->vext_a, 0, M * 8, st);
  if (vb) cudaMemcpyAsync(c->vext_b, vb, M * 8, cudaMemcpyDeviceToDevice, st); else cudaMemsetAsync(c->vext_b, 0, M * 8, st);
  if (de) cudaMemcpyAsync(c->dext, de, M * 16, cudaMemcpyDeviceToDevice, st); else cudaMemsetAsync(c->dext, 0, M * 16, st);
  return cuda_check(c, "set_external");
}

extern "C" wslda_status wslda_set_external_velocity(wslda_ctx* c, const double* va, const double* vb, void* stream) {
  if (!c) return WSLDA_EINVAL;
  if (!c->f.current_terms) return fail(c, WSLDA_ESTATE, "set_external_velocity: the context was created without current_terms");
  const int64_t M = c->P.M;
  cudaStream_t st = S(stream);
  if (va) cudaMemcpyAsync(c->cur_v, va, 3 * M * 8, cudaMemcpyDeviceToDevice, st); else cudaMemsetAsync(c->cur_v, 0, 3 * M * 8, st);
  if (vb) cudaMemcpyAsync(c->cur_v + 3 * M, vb, 3 * M * 8, cudaMemcpyDeviceToDevice, st); else cudaMemsetAsync(c->cur_v + 3 * M, 0, 3 * M * 8, st);
  LAUNCH(c, k_cur_w, nb(6 * M, 256), 256, 0, st, c->cur_A, c->cur_v, c->cur_W, 6 * M);
  return cuda_check(c, "set_external_velocity");
}

// ---- derivative engine: lap / grad of a batch of components (DerivArgs) -------------------------------------
static void deriv(wslda_ctx* c, const DerivArgs& a, cudaStream_t st) {
  const Plan& P = c->P;
  const int64_t M = P.M;
  int n_out = 0;
  for (int o = 0; o < 4; ++o) n_out += a.out[o] != nullptr;
  const double lgM = (double)(P.lg[0] + P.lg[1] + P.lg[2]);
  const double fl_fwd = 5.0 * M * lgM * a.ncomp, fl_x = 5.0 * M * P.lg[0] * a.ncomp, by_in = 16.0 * M * a.ncomp;
  if (P.onchip) {
    const size_t smem = (size_t)2 * P.G * M * 16;
    WORK(c, by_in, fl_fwd * (1 + n_out));
    LAUNCH(c, k_deriv_onchip, nb(a.ncomp, P.G), 256, smem, st, c->L, a, P.G);
    return;
  }
  const int64_t R = M / P.N[0];
  cplx* spec = c->scr[3];
  WORK(c, by_in, fl_fwd - fl_x);
  LAUNCH(c, k_planes_fwd, dim3(P.N[0] / P.PX, a.ncomp), 256, (size_t)P.PX * R * 16, st, c->L, a, spec, P.PX);
  WORK(c, 0, fl_x * (1 + n_out));
  LAUNCH(c, k_xlines, dim3((unsigned)(R >> P.lgT), a.ncomp), 256, (size_t)2 * P.N[0] * 16 << P.lgT, st, c->L, spec, a, P.lgT);
  OutList ol; int no = 0;
  for (int o = 0; o < 4; ++o) if (a.out[o]) ol.p[no++] = a.out[o];
  for (int o = no; o < 4; ++o) ol.p[o] = nullptr;
  WORK(c, 0, (fl_fwd - fl_x) * n_out);
  LAUNCH(c, k_planes_inv, dim3(P.N[0] / P.PX, a.ncomp, no), 256, (size_t)P.PX * R * 16, st, c->L, ol, P.PX);
}

// lap(alpha_sigma) of the current alpha fields (Eq. 40 needs it once per potential update)
static void update_lap_alpha(wslda_ctx* c, cudaStream_t st) {
  const int64_t M = c->P.M;
  cplx* in = c->scr[5];
  cplx* out = c->scr[6];
  if (c->P.chunk_n < 1) return;
  LAUNCH(c, k_real_to_cplx, nb(M, 256), 256, 0, st, c->alpha_a, c->alpha_b, in, M);
  DerivArgs a; memset(&a, 0, sizeof a);
  a.src = in; a.src_comp0 = 0; a.ncomp = 2; a.out[0] = out;
  deriv(c, a, st);
  LAUNCH(c, k_cplx_real_part, nb(M, 256), 256, 0, st, out, c->lap_a, c->lap_b, M);
}

extern "C" wslda_status wslda_set_potentials(wslda_ctx* c, const double* aa, const double* ab, const double* Ua,
                                             const double* Ub, const void* delta, void* stream) {
  if (!c || !aa || !ab || !Ua || !Ub || !delta) return fail(c, WSLDA_EINVAL, "set_potentials: null argument");
  const int64_t M = c->P.M;
  cudaStream_t st = S(stream);
  cudaMemcpyAsync(c->alpha_a, aa, M * 8, cudaMemcpyDeviceToDevice, st);
  cudaMemcpyAsync(c->alpha_b, ab, M * 8, cudaMemcpyDeviceToDevice, st);
  cudaMemcpyAsync(c->U_a, Ua, M * 8, cudaMemcpyDeviceToDevice, st);
  cudaMemcpyAsync(c->U_b, Ub, M * 8, cudaMemcpyDeviceToDevice, st);
  cudaMemcpyAsync(c->delta, delta, M * 16, cudaMemcpyDeviceToDevice, st);
  update_lap_alpha(c, st);
  return cuda_check(c, "set_potentials");
}

static void reduce_densities(wslda_ctx* c, cudaStream_t st);
static unsigned step_mask(const wslda_ctx* c);
static inline unsigned dens_group_of_field(int id) {
  return id <= WSLDA_F_RHO_B ? WSLDA_D_RHO : id <= WSLDA_F_TAU_B ? WSLDA_D_TAU : id == WSLDA_F_NU ? WSLDA_D_NU
       : id == WSLDA_F_BP ? WSLDA_D_BP : WSLDA_D_J;
}

extern "C" wslda_status wslda_set_reduce_hook(wslda_ctx* c, wslda_reduce_hook hook, void* user) {
  if (!c) return WSLDA_EINVAL;
  c->reduce_hook = hook; c->reduce_user = user;
  return WSLDA_OK;
}

extern "C" wslda_status wslda_get_field(wslda_ctx* c, int id, void* dst, void* stream) {
  if (!c || !dst) return fail(c, WSLDA_EINVAL, "get_field: null argument");
  const int64_t M = c->P.M;
  cudaStream_t st = S(stream);
  const void* src = nullptr; size_t bytes = M * 8;
  switch (id) {
    case WSLDA_F_ALPHA_A: src = c->alpha_a; break; case WSLDA_F_ALPHA_B: src = c->alpha_b; break;
    case WSLDA_F_U_A: src = c->U_a; break; case WSLDA_F_U_B: src = c->U_b; break;
    case WSLDA_F_LAP_ALPHA_A: src = c->lap_a; break; case WSLDA_F_LAP_ALPHA_B: src = c->lap_b; break;
    case WSLDA_F_LAMBDA_C: src = c->lambda; break; case WSLDA_F_G_EFF: src = c->geff; break;
    case WSLDA_F_V_A: src = c->V_a; break; case WSLDA_F_V_B: src = c->V_b; break;
    case WSLDA_F_DELTA: src = c->delta; bytes = M * 16; break;
    default: break;
  }
  if (id >= WSLDA_F_AA_X && id <= WSLDA_F_AB_Z) {
    if (c->f.current_terms) src = c->cur_A + (int64_t)(id - WSLDA_F_AA_X) * M;
    else { cudaMemsetAsync(dst, 0, bytes, st); return cuda_check(c, "get_field"); }
  }
  if (src) { cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, st); return cuda_check(c, "get_field"); }
  if (id < 0 || (id > WSLDA_F_JB_Z && id != WSLDA_F_BP)) return fail(c, WSLDA_EINVAL, "get_field: unknown field id");
  if (c->reduce_hook && (c->raw_local & (c->f.spin_symmetric ? (WSLDA_D_ALL | WSLDA_D_BP) : dens_group_of_field(id)))) reduce_densities(c, st);
  LAUNCH(c, k_get_density, nb(M, 256), 256, 0, st, c->raw, M, c->f.spin_symmetric, id, (double*)dst);
  return cuda_check(c, "get_field");
}

extern "C" wslda_status wslda_set_field(wslda_ctx* c, int id, const void* src, void* stream) {
  if (!c || !src) return fail(c, WSLDA_EINVAL, "set_field: null argument");
  const int64_t M = c->P.M;
  cudaStream_t st = S(stream);
  double* dst = nullptr;
  switch (id) {
    case WSLDA_F_RHO_A: dst = c->raw + DP_RHO_A * M; break; case WSLDA_F_RHO_B: dst = c->raw + DP_RHO_B * M; break;
    case WSLDA_F_TAU_A: dst = c->raw + DP_TAU_A * M; break; case WSLDA_F_TAU_B: dst = c->raw + DP_TAU_B * M; break;
    case WSLDA_F_LAMBDA_C: dst = c->lambda; c->lambda_valid = 1; break;
    case WSLDA_F_NU:   // interleaved complex -> two planes
      cudaMemcpy2DAsync(c->raw + DP_NU_RE * M, 8, src, 16, 8, M, cudaMemcpyDeviceToDevice, st);
      cudaMemcpy2DAsync(c->raw + DP_NU_IM * M, 8, (const char*)src + 8, 16, 8, M, cudaMemcpyDeviceToDevice, st);
      c->raw_local &= ~WSLDA_D_NU;
      return cuda_check(c, "set_field");
    default: return fail(c, WSLDA_EINVAL, "set_field: only raw rho/tau/nu and lambda_c can be set");
  }
  cudaMemcpyAsync(dst, src, M * 8, cudaMemcpyDeviceToDevice, st);
  if (id != WSLDA_F_LAMBDA_C) c->raw_local &= ~dens_group_of_field(id);     // the caller supplies whole-system densities
  return cuda_check(c, "set_field");
}

static wslda_status f3_apply_h(wslda_ctx* c, const cplx* psi, cplx* hpsi, double* eps_dev, int64_t n_first, int64_t n_count,
                               cudaStream_t st);

static wslda_status oc_apply_h(wslda_ctx* c, const cplx* psi, cplx* hpsi, double* eps_dev, int64_t n_first, int64_t n_count,
                               cudaStream_t st);

static Fields fields_of(const wslda_ctx* c) {
  Fields F;
  F.alpha_a = c->alpha_a; F.alpha_b = c->alpha_b; F.lap_a = c->lap_a; F.lap_b = c->lap_b; F.U_a = c->U_a; F.U_b = c->U_b;
  F.delta = c->delta; F.dext = c->dext; F.mu_a = c->mu_a; F.mu_b = c->mu_b;
  return F;
}

// H psi for the cnt spinors of a chunk: psi_chunk / scale_chunk (nullable) / out are already offset to the chunk's
// first spinor, n0 is its global index (per-spinor tables).  out is laid out [n - n0][2][M]; eps partials go to
// part_e.  Uses scr[0..3].
static void h_chunk(wslda_ctx* c, const cplx* psi_chunk, const double* scale_chunk, int64_t n0, int64_t cnt, cplx* out,
                    bool want_eps, cudaStream_t st) {
  const Plan& P = c->P;
  const int64_t M = P.M;
  const int kin = c->f.kin_form;
  DerivArgs a; memset(&a, 0, sizeof a);
  a.src = psi_chunk; a.src_comp0 = 0; a.ncomp = (int)(2 * cnt); a.scale = scale_chunk;
  cplx* cur = nullptr;
  if (c->f.current_terms) {                               // {W, grad} w first: scr[2] is free until the kinetic terms
    cur = c->scr[7];
    cplx* tmp = c->scr[2];
    const int64_t tot = 2 * cnt * M;
    for (int d = 0; d < P.nd; ++d) {
      const double* Wd = c->cur_W + (int64_t)d * M;      // W_a,d; W_b,d sits 3 M further
      DerivArgs g = a; g.out[1 + d] = tmp;
      deriv(c, g, st);
      LAUNCH(c, k_cur_acc, nb(tot, 256), 256, 0, st, cur, tmp, Wd, 3 * M, M, 2 * cnt, d == 0 ? 1 : 0);
      DerivArgs h = a; h.premul[0] = Wd; h.premul[1] = Wd + 3 * M; h.out[1 + d] = tmp;
      deriv(c, h, st);
      LAUNCH(c, k_cur_acc, nb(tot, 256), 256, 0, st, cur, tmp, (const double*)nullptr, 0, M, 2 * cnt, 0);
    }
  }
  if (kin == WSLDA_KIN_DIVGRAD) {
    for (int d = 0; d < P.nd; ++d) a.out[1 + d] = c->scr[d];
    deriv(c, a, st);
    for (int d = 0; d < P.nd; ++d) {                    // s_d <- d_d (alpha s_d), in place
      DerivArgs b; memset(&b, 0, sizeof b);
      b.src = c->scr[d]; b.src_comp0 = 0; b.ncomp = a.ncomp; b.premul[0] = c->alpha_a; b.premul[1] = c->alpha_b;
      b.out[1 + d] = c->scr[d];
      deriv(c, b, st);
    }
  } else {
    a.out[0] = c->scr[0];
    deriv(c, a, st);
    if (kin == WSLDA_KIN_SYM40) {
      DerivArgs b = a;
      b.premul[0] = c->alpha_a; b.premul[1] = c->alpha_b; b.out[0] = c->scr[1];
      deriv(c, b, st);
    }
  }
  WORK(c, 64.0 * M * cnt, 0);      // reads psi, writes H psi
  LAUNCH(c, k_hmix, dim3(P.nblk, (unsigned)cnt), P.pt_threads, 0, st, psi_chunk, scale_chunk, c->kperp2 + n0, kin, P.nd,
         c->scr[0], c->scr[1], c->scr[2], fields_of(c), M, out, want_eps ? c->part_e : nullptr, P.nblk, (const cplx*)cur);
}

extern "C" wslda_status wslda_apply_h(wslda_ctx* c, const void* psi_, void* hpsi_, double* eps_dev, int64_t n_first,
                                      int64_t n_count, void* stream) {
  if (!c || !psi_ || !hpsi_ || psi_ == hpsi_) return fail(c, WSLDA_EINVAL, "apply_h: null or aliased buffers");
  if (n_first < 0 || n_count < 0 || n_first + n_count > c->P.n_wf) return fail(c, WSLDA_EINVAL, "apply_h: spinor range out of bounds");
  const cplx* psi = (const cplx*)psi_; cplx* hpsi = (cplx*)hpsi_;
  const int64_t M = c->P.M;
  cudaStream_t st = S(stream);
  if (c->P.fast || c->P.f6) return f3_apply_h(c, psi, hpsi, eps_dev, n_first, n_count, st);
  if (c->P.oc) return oc_apply_h(c, psi, hpsi, eps_dev, n_first, n_count, st);
  for (int64_t n0 = n_first; n0 < n_first + n_count; n0 += c->P.chunk_n) {
    const int64_t cnt = (n_first + n_count - n0 < c->P.chunk_n) ? n_first + n_count - n0 : c->P.chunk_n;
    h_chunk(c, psi + 2 * n0 * M, nullptr, n0, cnt, hpsi + 2 * n0 * M, true, st);
    LAUNCH(c, k_from_partials, nb(cnt * 32, 128), 128, 0, st, c->part_e, c->P.nblk, cnt, c->dV, 0, c->eps + n0,
           eps_dev ? eps_dev + n0 : nullptr);
  }
  return cuda_check(c, "apply_h");
}

// densities of the cnt spinors of a chunk (psi_chunk / scale_chunk already offset, n0 = global index of the
// first), added into the raw sums (accumulate) or overwriting the selected planes.  Uses scr[0..3].
static void dens_chunk(wslda_ctx* c, const cplx* psi_chunk, const double* scale_chunk, int64_t n0, int64_t cnt,
                       unsigned mask, int accumulate, cudaStream_t st) {
  const Plan& P = c->P;
  const int64_t M = P.M;
  DensArgs d; memset(&d, 0, sizeof d);
  if (mask & (WSLDA_D_TAU | WSLDA_D_J | WSLDA_D_BP)) {
    DerivArgs a; memset(&a, 0, sizeof a);
    a.src = psi_chunk; a.src_comp0 = 0; a.ncomp = (int)(2 * cnt); a.scale = scale_chunk;
    if (mask & (WSLDA_D_TAU | WSLDA_D_J)) for (int k = 0; k < P.nd; ++k) { a.out[1 + k] = c->scr[k]; d.grad[k] = c->scr[k]; }
    if (mask & WSLDA_D_BP) { a.out[0] = c->scr[5]; d.lap = c->scr[5]; }      // Laplacians for B' (Eq. 68)
    deriv(c, a, st);
  }
  int64_t G = P.dG < cnt ? P.dG : cnt;
  const int64_t per = (cnt + G - 1) / G;
  G = (cnt + per - 1) / per;
  d.psi = psi_chunk; d.scale = scale_chunk; d.cpref = c->cpref + n0; d.kperp2 = c->kperp2 + n0;
  d.w_a = c->w_a + n0; d.w_b = c->w_b + n0; d.nd = P.nd; d.M = M; d.n_count = cnt; d.per_group = per; d.mask = mask;
  WORK(c, 32.0 * M * cnt, 0);
  LAUNCH(c, k_density, dim3(P.nblk, (unsigned)G), P.pt_threads, 0, st, d, c->dpart);
  if (G > 16) LAUNCH(c, k_density_reduce_wide, dim3(nb(M, 8), DP_COUNT), 256, 0, st, c->dpart, (int)G, c->raw, M, mask, accumulate);
  else LAUNCH(c, k_density_reduce, dim3(nb(M, 256), DP_COUNT), 256, 0, st, c->dpart, (int)G, c->raw, M, mask, accumulate);
}

// tau and j of spinors [n_first, n_first + n_count) on a cubic 32^3 / 64^3 lattice, axis by axis (gdens.cuh)
static bool gdens_ok(const wslda_ctx* c) {
  const Plan& P = c->P;
  return P.nd == 3 && P.N[0] == P.N[1] && P.N[1] == P.N[2] && (P.N[0] == 32 || P.N[0] == 64) && !g_tune.disable_axis_split;
}
static void gdens(wslda_ctx* c, const cplx* psi, int64_t n_first, int64_t n_count, unsigned mask, int accumulate, cudaStream_t st,
                  const double* scale = nullptr) {
  const Plan& P = c->P;
  const int N = P.N[0];
  const int64_t M = P.M;
  GdArgs a;
  a.psi = psi + 2 * n_first * M; a.cpref = c->cpref + n_first; a.w_a = c->w_a + n_first; a.w_b = c->w_b + n_first;
  a.scale = scale ? scale + n_first : nullptr;
  const double PI = 3.14159265358979323846264338327950288;
  for (int d = 0; d < 3; ++d) {
    const double len = N * c->dx[d];
    for (int j = 0; j < 64; ++j) a.kd[d][j] = (j >= N || j == N / 2) ? 0.0 : (j < N / 2 ? 2.0 * PI * j / len : 2.0 * PI * (j - N) / len);
  }
  a.part = c->dpart; a.n = (int)n_count;
  int G = P.dG;                                          // the partial planes share the general path's buffer: G x 12 planes
  if (G > n_count) G = (int)n_count;
  if (G < 1) G = 1;
  a.G = G;
  const int tiles = N * N / (N == 32 ? 128 : 64);
  const double lines = 3.0 * 2.0 * (double)N * N * (double)n_count;
  WORK(c, 32.0 * M * n_count, lines * 2.0 * 5.0 * N * P.lg[0]);
  // (k_gdens_reduce only reads the planes of `mask`: a variant that skips the other kind leaves its partial planes stale)
  const int what = ((mask & WSLDA_D_TAU) ? 1 : 0) | ((mask & WSLDA_D_J) ? 2 : 0);
  void (*k)(GdArgs) = N == 32 ? (what == 1 ? k_gdens<32, 1> : what == 2 ? k_gdens<32, 2> : k_gdens<32, 3>)
                              : (what == 1 ? k_gdens<64, 1> : what == 2 ? k_gdens<64, 2> : k_gdens<64, 3>);
  LAUNCHN(c, "k_gdens", k, dim3(tiles, 6, G), 128, 2 * 32 * 128 * 8, st, a);
  LAUNCH(c, k_gdens_reduce, nb(M, 256), 256, 0, st, c->dpart, G, M, c->raw, mask, accumulate);
}

// B' (Eq. 68) of the same range the same way: second derivatives axis by axis (gdens.cuh)
static void gdens_bp(wslda_ctx* c, const cplx* psi, int64_t n_first, int64_t n_count, int accumulate, cudaStream_t st,
                     const double* scale = nullptr) {
  const Plan& P = c->P;
  const int N = P.N[0];
  const int64_t M = P.M;
  GdArgs a;
  a.psi = psi + 2 * n_first * M; a.cpref = c->cpref + n_first; a.w_a = c->w_a + n_first; a.w_b = c->w_b + n_first;
  a.scale = scale ? scale + n_first : nullptr;
  for (int d = 0; d < 3; ++d)
    for (int j = 0; j < 64; ++j) a.kd[d][j] = j < N ? c->hk2[d][j] : 0.0;       // squared wave numbers, Nyquist mode kept
  a.part = c->dpart; a.n = (int)n_count;
  int G = P.dG;
  if (G > n_count) G = (int)n_count;
  if (G < 1) G = 1;
  a.G = G;
  const int tiles = N * N / (N == 32 ? 128 : 64);
  WORK(c, 32.0 * M * n_count, 3.0 * 2.0 * (double)N * N * (double)n_count * 2.0 * 5.0 * N * P.lg[0]);
  if (N == 32) LAUNCHN(c, "k_gdens_bp", k_gdens_bp<32>, dim3(tiles, 6, G), 128, 2 * 32 * 128 * 8, st, a);
  else LAUNCHN(c, "k_gdens_bp", k_gdens_bp<64>, dim3(tiles, 6, G), 128, 2 * 32 * 128 * 8, st, a);
  LAUNCH(c, k_gdens_bp_reduce, nb(M, 256), 256, 0, st, c->dpart, G, M, c->raw, accumulate);
}

extern "C" wslda_status wslda_densities(wslda_ctx* c, const void* psi_, int64_t n_first, int64_t n_count, unsigned mask,
                                        int accumulate, void* stream) {
  if (!c || !psi_) return fail(c, WSLDA_EINVAL, "densities: null argument");
  if (n_first < 0 || n_count < 0 || n_first + n_count > c->P.n_wf) return fail(c, WSLDA_EINVAL, "densities: spinor range out of bounds");
  if (!mask || (mask & ~(WSLDA_D_ALL | WSLDA_D_BP))) return fail(c, WSLDA_EINVAL, "densities: bad which_mask");
  if (c->reduce_hook && accumulate && (mask & ~c->raw_local)) return fail(c, WSLDA_EINVAL, "densities: accumulate onto a block already summed over the ranks");
  c->raw_local |= mask;
  cudaStream_t st = S(stream);
  if (n_count == 0 && !accumulate) {
    LAUNCH(c, k_density_reduce, dim3(nb(c->P.M, 256), DP_COUNT), 256, 0, st, c->dpart, 0, c->raw, c->P.M, mask, 0);
  }
  if (n_count > 0 && (mask & (WSLDA_D_TAU | WSLDA_D_J)) && gdens_ok(c)) {     // cubic 32^3 / 64^3: gradients axis by axis
    gdens(c, (const cplx*)psi_, n_first, n_count, mask & (WSLDA_D_TAU | WSLDA_D_J), accumulate, st);
    mask &= ~(WSLDA_D_TAU | WSLDA_D_J);
    if (!mask) return cuda_check(c, "densities");
  }
  if (n_count > 0 && (mask & WSLDA_D_BP) && gdens_ok(c)) {                     // B' by second derivatives axis by axis
    gdens_bp(c, (const cplx*)psi_, n_first, n_count, accumulate, st);
    mask &= ~WSLDA_D_BP;
    if (!mask) return cuda_check(c, "densities");
  }
  // without gradient fields no scratch is involved: the whole range is one "chunk" (one k_density launch)
  const int64_t step = (mask & (WSLDA_D_TAU | WSLDA_D_J | WSLDA_D_BP)) ? c->P.chunk_n : (n_count > 0 ? n_count : 1);
  for (int64_t n0 = n_first; n0 < n_first + n_count; n0 += step) {
    const int64_t cnt = (n_first + n_count - n0 < step) ? n_first + n_count - n0 : step;
    dens_chunk(c, (const cplx*)psi_ + 2 * n0 * c->P.M, nullptr, n0, cnt, mask, (accumulate || n0 > n_first) ? 1 : 0, st);
  }
  return cuda_check(c, "densities");
}

// Sharded runs (wslda_set_reduce_hook): the density block holds this rank's partial sums until the hook has summed it
// over the ranks; every potential is formed from the reduced block.
// raw_local is the set of density groups (WSLDA_D_* bits) whose planes hold LOCAL sums: only those are handed to the
// hook -- a plane that is already a whole-system sum (tau and j left by an earlier wslda_densities while a step rebuilds
// rho and nu only) must not be summed again.  The groups' planes are contiguous in the order RHO, NU, TAU, J, so the
// dirty groups are reduced as maximal contiguous runs (one hook call for rho + nu inside a step).
static void reduce_densities(wslda_ctx* c, cudaStream_t st) {
  if (c->reduce_hook) {
    static const unsigned grp[5] = {WSLDA_D_RHO, WSLDA_D_NU, WSLDA_D_TAU, WSLDA_D_J, WSLDA_D_BP};
    static const int first[6] = {DP_RHO_A, DP_NU_RE, DP_TAU_A, DP_JA0, DP_BP_RE, DP_COUNT};
    int g = 0;
    while (g < 5) {
      if (!(c->raw_local & grp[g])) { ++g; continue; }
      int h = g;
      while (h + 1 < 5 && (c->raw_local & grp[h + 1])) ++h;
      c->reduce_hook(c->reduce_user, c->raw + (int64_t)first[g] * c->P.M, (int64_t)(first[h + 1] - first[g]) * c->P.M, (void*)st);
      g = h + 1;
    }
  }
  c->raw_local = 0;
}

static wslda_status observables(wslda_ctx* c, double* obs_dev, const double* ref_dev, double tol_n, double tol_e, cudaStream_t st,
                                const char* where);
// Eqs. 66-70 on top of the potentials just built: N from the observables kernel, div j_sigma by six
// field derivatives (one per spin and held axis, Nyquist rule of an odd derivative), then the pointwise k_qf.
static void quantum_friction(wslda_ctx* c, const FuncParams& fp, cudaStream_t st) {
  const int64_t M = c->P.M;
  observables(c, nullptr, nullptr, 0.0, 0.0, st, "quantum friction");
  cplx* in = c->scr[5];
  cplx* out = c->scr[6];
  for (int d = 0; d < c->P.nd; ++d) {
    LAUNCH(c, k_j_to_cplx, nb(M, 256), 256, 0, st, c->raw, d, c->f.spin_symmetric, in, M);
    DerivArgs a; memset(&a, 0, sizeof a);
    a.src = in; a.src_comp0 = 0; a.ncomp = 2; a.out[1 + d] = out;
    deriv(c, a, st);
    LAUNCH(c, k_real_acc, nb(2 * M, 256), 256, 0, st, c->qf_divj, out, 2 * M, d == 0 ? 1 : 0);
  }
  LAUNCH(c, k_qf, nb(M, 256), 256, 0, st, fp, c->raw, c->qf_divj, c->obs_out, c->V_a, c->V_b, c->U_a, c->U_b, c->delta, M);
}

// fresh: the block was just rebuilt from this rank's spinors (every call inside a step)
static void potentials(wslda_ctx* c, cudaStream_t st, bool fresh) {
  if (c->f.func_id == WSLDA_FUNC_FIXED) return;
  if (fresh) c->raw_local |= step_mask(c);               // the planes the step has just rebuilt from this rank's spinors
  if (c->raw_local) reduce_densities(c, st);
  const int64_t M = c->P.M;
  FuncParams fp;
  fp.func_id = c->f.func_id; fp.force_a1 = c->f.force_a1; fp.spin_symmetric = c->f.spin_symmetric;
  fp.current_terms = c->f.current_terms; fp.quantum_friction = c->f.quantum_friction;
  fp.qf_alpha = c->f.qf_alpha; fp.qf_beta = c->f.qf_beta; fp.qf_gamma = c->f.qf_gamma; fp.qf_rho0 = c->f.qf_rho0; fp.qf_nreq = c->f.qf_nreq;
  fp.four_pi_as = c->f.four_pi_as; fp.C = c->f.C; fp.E_cut = c->f.E_cut; fp.rho_floor = c->f.rho_floor;
  fp.mu_a = c->mu_a; fp.mu_b = c->mu_b;
  const int frozen = c->f.lambda_mode == 1 && c->lambda_valid;
  LAUNCH(c, k_potentials, nb(M, 128), 128, 0, st, fp, c->raw, c->vext_a, c->vext_b, frozen, c->alpha_a, c->alpha_b, c->V_a,
         c->V_b, c->U_a, c->U_b, c->lambda, c->geff, c->delta, M, c->cur_A, c->cur_v, c->cur_W);
  c->lambda_valid = 1;
  if (c->f.kin_form == WSLDA_KIN_SYM40 && c->f.func_id == WSLDA_FUNC_ASLDA && !c->f.force_a1) update_lap_alpha(c, st);
  if (c->f.quantum_friction) quantum_friction(c, fp, st);
}

// observables from the density block as it stands (Eqs. 33a-g); ref != null adds the device-side conservation check
static wslda_status observables(wslda_ctx* c, double* obs_dev, const double* ref_dev, double tol_n, double tol_e, cudaStream_t st,
                                const char* where) {
  const int64_t M = c->P.M;
  if (c->reduce_hook && c->raw_local) reduce_densities(c, st);
  ObsArgs a;
  a.P.func_id = c->f.func_id; a.P.force_a1 = c->f.force_a1; a.P.spin_symmetric = c->f.spin_symmetric;
  a.P.current_terms = c->f.current_terms; a.P.four_pi_as = c->f.four_pi_as; a.P.C = c->f.C; a.P.E_cut = c->f.E_cut;
  a.P.rho_floor = c->f.rho_floor; a.P.mu_a = c->mu_a; a.P.mu_b = c->mu_b;
  a.raw = c->raw; a.alpha_a = c->alpha_a; a.alpha_b = c->alpha_b; a.vext_a = c->vext_a; a.vext_b = c->vext_b;
  a.cur_v = c->cur_v; a.delta = c->delta; a.dext = c->dext; a.dVf = c->dV * c->Lperp; a.M = M;
  const int nblk = (int)((M + 255) / 256);
  LAUNCH(c, k_energy, nblk, 256, 0, st, a, c->obs_part);
  LAUNCH(c, k_energy_final, 1, 32, 0, st, c->obs_part, nblk, c->obs_out, ref_dev, tol_n, tol_e, ref_dev ? c->wd_flag : (int*)nullptr);
  if (obs_dev) cudaMemcpyAsync(obs_dev, c->obs_out, WS_NOBS * sizeof(double), cudaMemcpyDeviceToDevice, st);
  if (ref_dev && c->err_host) cudaMemcpyAsync(c->err_host + 1, c->wd_flag, sizeof(int), cudaMemcpyDeviceToHost, st);
  return cuda_check(c, where);
}

extern "C" wslda_status wslda_energy(wslda_ctx* c, double* obs_dev, void* stream) {
  if (!c || !obs_dev) return fail(c, WSLDA_EINVAL, "energy: null argument");
  return observables(c, obs_dev, nullptr, 0.0, 0.0, S(stream), "energy");
}

extern "C" wslda_status wslda_watchdog(wslda_ctx* c, const double* ref_dev, double tol_number, double tol_energy, double* obs_dev,
                                       void* stream) {
  if (!c || !ref_dev) return fail(c, WSLDA_EINVAL, "watchdog: null argument");
  if (!(tol_number >= 0) || !(tol_energy >= 0)) return fail(c, WSLDA_EINVAL, "watchdog: tolerances must be >= 0");
  return observables(c, obs_dev, ref_dev, tol_number, tol_energy, S(stream), "watchdog");
}

// ---- the FP64 denominator of the roofline: a dependent-chain DFMA probe (8 independent chains per thread, 16 warps per
// SM scheduler's worth of threads), timed with CUDA events; reports 2 flops per DFMA ----------------------------------------
__global__ void __launch_bounds__(256) k_fp64_probe(double* out, int iters, double a, double b) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0, x4 = x0 + 4.0, x5 = x0 + 5.0, x6 = x0 + 6.0, x7 = x0 + 7.0;
  for (int i = 0; i < iters; ++i) {
    x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
    x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
  }
  const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 123.456) out[0] = s;                             // never true: keeps the chains alive
}
extern "C" wslda_status wslda_fp64_probe(double* flops_per_s, double* sm_count_out) {
  if (!flops_per_s) return WSLDA_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
    snprintf(g_err, 256, "fp64_probe: no CUDA device"); return WSLDA_ECUDA;
  }
  double* d = nullptr;
  if (cudaMalloc(&d, 8) != cudaSuccess) { snprintf(g_err, 256, "fp64_probe: cudaMalloc failed"); return WSLDA_ECUDA; }
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = sms * 8, iters = 1 << 15;
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {                       // first repetition warms up; keep the best of the rest
    cudaEventRecord(e0);
    k_fp64_probe<<<blocks, 256>>>(d, iters, 0.999999, 1e-9);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
    const double f = 2.0 * 8.0 * (double)iters * 256.0 * blocks / (ms * 1e-3);
    if (rep > 0 && f > best) best = f;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  if (cudaGetLastError() != cudaSuccess) { snprintf(g_err, 256, "fp64_probe: CUDA error"); return WSLDA_ECUDA; }
  *flops_per_s = best;
  if (sm_count_out) *sm_count_out = (double)sms;
  return WSLDA_OK;
}

extern "C" wslda_status wslda_update_potentials(wslda_ctx* c, void* stream) {
  if (!c) return WSLDA_EINVAL;
  potentials(c, S(stream), false);
  return cuda_check(c, "update_potentials");
}
