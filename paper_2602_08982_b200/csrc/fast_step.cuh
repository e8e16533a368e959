// fast_step.cuh -- host side of the fused 3-D path (fast3d.cuh): H psi in three passes per chunk, and the
// Alg. 2 step as chunk pipelines on up to four concurrent streams so that the passes of
// different chunks overlap (HBM-bound, L2-bound and FP64-bound phases run side by side on the SMs).
#pragma once
#include "onchip_step.cuh"

static F3Fields f3_fields(const wslda_ctx* c) {
  F3Fields F;
  F.alpha[0] = c->alpha_a; F.alpha[1] = c->alpha_b; F.lap[0] = c->lap_a; F.lap[1] = c->lap_b;
  F.U[0] = c->U_a; F.U[1] = c->U_b; F.delta = c->delta; F.dext = c->dext; F.mu[0] = c->mu_a; F.mu[1] = c->mu_b;
  return F;
}

// persistent grids: at most (CTAs per SM) x 148 SMs, warps stride over the items
static inline int f3_grid(int want, int per_sm) { const int cap = per_sm * 148; return want < cap ? want : cap; }

// out = APPLY: H psi | CORR: C_part - i kappa H psi | RHS: -i H psi  for the cnt spinors of a chunk (psi_chunk,
// scale_chunk, out, cpart already offset to the chunk; n0 = global index of its first spinor); pass-C partial
// sums go to f_part[q].  q = scratch slot, st = the stream that owns it.
static void f3_hpsi(wslda_ctx* c, int q, cudaStream_t st, const cplx* psi_chunk, const double* scale_chunk, int64_t n0,
                    int cnt, int mode, cplx* out, const cplx* cpart, double kappa) {
  const Plan& P = c->P;
  const int NX = P.N[0];
  const int64_t M = P.M;
  const bool sym = c->f.kin_form == WSLDA_KIN_SYM40;
  const int nspec = sym ? 2 : 1;
  const double fl_plane = 5.0 * M * 10.0 * 2 * cnt * nspec, fl_x = 5.0 * M * P.lg[0] * 2.0 * 2 * cnt * nspec;
  F3PassA a;
  a.psi = psi_chunk; a.scale = scale_chunk; a.alpha[0] = c->alpha_a; a.alpha[1] = c->alpha_b;
  a.spec0 = c->f_spec0[q]; a.spec1 = c->f_spec1[q]; a.n_items = cnt * 2 * NX; a.NX = NX;
  WORK(c, 32.0 * M * cnt, fl_plane);                       // reads psi once
  auto ka = sym ? k_f3_pass_a<true> : k_f3_pass_a<false>;
  LAUNCHN(c, "k_f3_pass_a", ka, f3_grid((a.n_items + 3) / 4, 3), 128, 4 * F3_TILE_BYTES, st, a);
  F3PassB b;
  b.spec[0] = c->f_spec0[q]; b.spec[1] = c->f_spec1[q]; b.n_spec = nspec; b.n_items = cnt * 2 * F3_N;
  b.ky2 = c->k2n[1]; b.kz2 = c->k2n[2]; b.invM = c->L.invM;
  for (int j = 0; j < 32; ++j) b.kx2[j] = j < NX ? c->hk2[0][j] : 0.0;
  WORK(c, 0, fl_x);
  auto kb = NX == 32 ? k_f3_pass_b<32> : NX == 16 ? k_f3_pass_b<16> : k_f3_pass_b<8>;
  LAUNCHN(c, "k_f3_pass_b", kb, f3_grid((b.n_items + 3) / 4, 3), 128, 0, st, b);
  F3PassC k;
  k.spec0 = c->f_spec0[q]; k.spec1 = c->f_spec1[q]; k.psi = psi_chunk; k.scale = scale_chunk; k.kperp2 = c->kperp2 + n0;
  k.F = f3_fields(c); k.out = out; k.cpart = cpart; k.kappa = kappa; k.part = c->f_part[q]; k.n_items = cnt * NX; k.NX = NX;
  const int grid = f3_grid((k.n_items + 1) / 2, sym ? 3 : 6);
  const size_t sm_sym = 2 * (F3_TILE_BYTES + F3_PLANE * 16), sm_lap = 2 * F3_TILE_BYTES;
  WORK(c, mode == F3_CORR ? 32.0 * M * cnt : (mode == F3_APPLY ? 32.0 * M * cnt : 0.0), fl_plane);
  void (*kc)(F3PassC);
  if (sym) kc = mode == F3_APPLY ? k_f3_pass_c<true, F3_APPLY> : mode == F3_CORR ? k_f3_pass_c<true, F3_CORR> : k_f3_pass_c<true, F3_RHS>;
  else kc = mode == F3_APPLY ? k_f3_pass_c<false, F3_APPLY> : mode == F3_CORR ? k_f3_pass_c<false, F3_CORR> : k_f3_pass_c<false, F3_RHS>;
  LAUNCHN(c, "k_f3_pass_c", kc, grid, 64, sym ? sm_sym : sm_lap, st, k);
}

// One persistent dataflow launch (mega3d.cuh) over spinors [n0, n0 + n) of the caller's buffers:
// APPLY: out = H psi (+ eps via k_f3_scal); CORR: psi buffer <- phi_new (normalised) + densities; RHS: out = f(psi).
static bool f3_uses_t3(const wslda_ctx* c) { return c->t3 && c->f.kin_form == WSLDA_KIN_SYM40; }
static void f3_mega(wslda_ctx* c, cudaStream_t st, int mode, const cplx* psi, const double* scale, int64_t n0, int64_t n,
                    cplx* out, const cplx* cpart, double kappa, int do_dens, double* eps_user = nullptr) {
  const Plan& P = c->P;
  const bool sym = c->f.kin_form == WSLDA_KIN_SYM40;
  F3Mega a;
  a.psi = psi; a.scale = scale; a.kperp2 = c->kperp2 + n0; a.F = f3_fields(c);
  a.ky2 = c->k2n[1]; a.kz2 = c->k2n[2];
  for (int j = 0; j < 32; ++j) a.kx2[j] = j < P.N[0] ? c->hk2[0][j] : 0.0;
  a.invM = c->L.invM; a.dV = c->dV; a.kappa = kappa;
  a.spec0 = c->m_spec0; a.spec1 = c->m_spec1; a.X = c->m_X; a.out = out; a.cpart = cpart; a.part = c->m_part;
  a.eps_out = mode == F3_APPLY ? nullptr : c->eps + n0;
  a.use_shift = c->f.subtract_mean_energy; a.normalize = c->f.normalize; a.do_dens = do_dens;
  a.cpref = c->cpref + n0; a.w_a = c->w_a + n0; a.w_b = c->w_b + n0; a.acc = c->m_acc; a.sync = c->m_sync;
  a.n = (int)n; a.gs = P.gs; a.G = (int)((n + P.gs - 1) / P.gs); a.NX = P.N[0];
  cudaMemsetAsync(c->m_sync, 0, sizeof(F3Sync) + (size_t)4 * a.G * sizeof(int), st);
  a.pack = c->m_pack;
  LAUNCH(c, k_f3_pack, nb(P.M, 256), 256, 0, st, a.F, sym ? 1 : 0, P.M, c->m_pack);
  const int NX = P.N[0], nspec = sym ? 2 : 1;
  const int IT = a.gs * 2 * NX / 4 + a.gs * 16 + (sym ? a.gs * NX : a.gs * NX / 2) + (mode == F3_APPLY ? 0 : NX * F3_DSPLIT);
  const long total = (long)(a.G + 3) * IT;
  const int grid = (int)(total < c->mega_grid ? total : c->mega_grid);
  const double M = (double)P.M;
  WORK(c, M * n * (mode == F3_CORR ? 96.0 : 64.0), 5.0 * M * (P.lg[0] + 10.0) * 2.0 * 2 * nspec * n);
  void (*k)(F3Mega);
  if (sym) k = mode == F3_APPLY ? k_f3_mega<true, F3_APPLY> : mode == F3_CORR ? k_f3_mega<true, F3_CORR> : k_f3_mega<true, F3_RHS>;
  else k = mode == F3_APPLY ? k_f3_mega<false, F3_APPLY> : mode == F3_CORR ? k_f3_mega<false, F3_CORR> : k_f3_mega<false, F3_RHS>;
  if (f3_uses_t3(c)) {                                     // 32^3 Eq. 40: warp-specialised, TMA-fed (mega3t.cuh)
    T3Maps maps = c->t3_maps;
    if (!t3_encode_cplx(&maps.psiP, &maps.psiX, psi, (size_t)2 * n)) { snprintf(c->err, 256, "cuTensorMapEncodeTiled failed (psi)"); c->sticky = 1; return; }
    T3Mega A;
    A.m = a; A.m.sync = nullptr; A.sync = (T3Sync*)c->m_sync; A.sn_out = c->scale2 + n0;
    A.m.eps_out = c->eps + n0; A.eps_user = eps_user;
    for (int j = 0; j < 32; ++j) { A.k2all[j] = c->hk2[2][j]; A.k2all[32 + j] = c->hk2[1][j]; A.k2all[64 + j] = c->hk2[0][j]; }
    A.gs = c->t3_gs; A.r = c->t3_r; A.R = c->t3_ring; A.RA = F3_RING; A.lag = c->t3_lag; A.G = (int)((n + A.gs - 1) / A.gs); A.spin_limit = c->spin_limit;
    A.m.gs = A.gs; A.m.G = A.G;
    cudaMemsetAsync(c->m_sync, 0, sizeof(T3Sync) + ((size_t)3 * ((n + A.r - 1) / A.r) + (size_t)2 * A.G) * sizeof(int), st);
    void (*kt)(T3Maps, T3Mega) = mode == F3_APPLY ? k_t3_mega<F3_APPLY> : mode == F3_CORR ? k_t3_mega<F3_CORR> : k_t3_mega<F3_RHS>;
    LAUNCHN(c, mode == F3_APPLY ? "k_t3_mega_apply" : mode == F3_CORR ? "k_t3_mega_corr" : "k_t3_mega_rhs", kt, c->t3_grid, T3_THREADS,
            T3_SMEM_BYTES, st, maps, A);
    cudaMemcpyAsync(c->err_host, &A.sync->error, sizeof(int), cudaMemcpyDeviceToHost, st);      // read at the next API call
    return;
  }
  if (c->dm3 && sym) {                       // 32^3 Eq. 40: matrix-form line derivatives on DMMA (mega3m.cuh)
    F3MMega A;
    A.m = a; A.pm = c->sep_pm; A.em = c->sep_em; A.mat = c->m_mat; A.mat1 = c->m_mat + 1536; A.curW = c->f.current_terms ? c->cur_W : nullptr;
    const int ITs = a.gs * 32 / A.pm + a.gs * 32 / A.em + (mode == F3_APPLY ? 0 : 32 * F3_DSPLIT);
    const long tot = (long)(a.G + 2) * ITs;
    const int cap = c->f.current_terms ? c->dm3_grid_cur : c->dm3_grid;
    const int gr = (int)(tot < cap ? tot : cap);
    void (*km)(F3MMega) = mode == F3_APPLY ? k_f3m_mega<F3_APPLY> : mode == F3_CORR ? k_f3m_mega<F3_CORR> : k_f3m_mega<F3_RHS>;
    if (c->f.current_terms)                                // the coupling of Eq. 4c inside the matrix-form kernels (own instantiation, 2 CTAs per SM)
      km = mode == F3_APPLY ? k_f3m_mega<F3_APPLY, true> : mode == F3_CORR ? k_f3m_mega<F3_CORR, true> : k_f3m_mega<F3_RHS, true>;
    LAUNCHN(c, mode == F3_APPLY ? "k_f3m_mega_apply" : mode == F3_CORR ? "k_f3m_mega_corr" : "k_f3m_mega_rhs", km, gr, 128, F3M_BUF_BYTES, st, A);
    cudaMemcpyAsync(c->err_host, &c->m_sync->error, sizeof(int), cudaMemcpyDeviceToHost, st);
    return;
  }
  if (c->sep3) {                             // 32^3: axis-by-axis Laplacian, two passes (mega3s.cuh)
    F3SMega A;
    A.m = a; A.pm = c->sep_pm; A.em = c->sep_em;
    for (int j = 0; j < 32; ++j) { A.k2zy[j] = c->hk2[2][j]; A.k2zy[32 + j] = c->hk2[1][j]; }
    const int ITs = a.gs * (sym ? 32 : 16) / A.pm + a.gs * 16 / A.em + (mode == F3_APPLY ? 0 : 32 * F3_DSPLIT);
    const long tot = (long)(a.G + 2) * ITs;
    const int gr = (int)(tot < c->mega_grid ? tot : c->mega_grid);
    void (*ks)(F3SMega);
    if (sym) ks = mode == F3_APPLY ? k_f3s_mega<true, F3_APPLY> : mode == F3_CORR ? k_f3s_mega<true, F3_CORR> : k_f3s_mega<true, F3_RHS>;
    else ks = mode == F3_APPLY ? k_f3s_mega<false, F3_APPLY> : mode == F3_CORR ? k_f3s_mega<false, F3_CORR> : k_f3s_mega<false, F3_RHS>;
    LAUNCHN(c, mode == F3_APPLY ? "k_f3s_mega_apply" : mode == F3_CORR ? "k_f3s_mega_corr" : "k_f3s_mega_rhs", ks, gr, 128,
            4 * F3_TILE_BYTES, st, A);
    cudaMemcpyAsync(c->err_host, &c->m_sync->error, sizeof(int), cudaMemcpyDeviceToHost, st);
    return;
  }
  LAUNCHN(c, mode == F3_APPLY ? "k_f3_mega_apply" : mode == F3_CORR ? "k_f3_mega_corr" : "k_f3_mega_rhs", k, grid, 128,
          4 * F3_TILE_BYTES, st, a);
  cudaMemcpyAsync(c->err_host, &c->m_sync->error, sizeof(int), cudaMemcpyDeviceToHost, st);
}

// ---- 64^3 (mega64.cuh) -------------------------------------------------------------------------------------------
// eps_n from the per-(component, x-plane) partial sums of an APPLY launch: one warp per spinor
__global__ void k_f6_scal(const double* part, int n, double dV, double* eps, double* eps_user) {
  const int s = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (s >= n) return;
  const double* pp = part + (size_t)(2 * s) * F6_N;
  double t = (pp[lane] + pp[32 + lane]) + (pp[64 + lane] + pp[96 + lane]);
  t = warp_sum(t);
  if (lane == 0) { eps[s] = dV * t; if (eps_user) eps_user[s] = dV * t; }
}

static void f6_mega(wslda_ctx* c, cudaStream_t st, int mode, const cplx* psi, const double* scale, int64_t n0, int64_t n,
                    cplx* out, const cplx* cpart, double kappa, int do_dens) {
  const Plan& P = c->P;
  F6Mega a;
  a.psi = psi; a.scale = scale; a.kperp2 = c->kperp2 + n0; a.F = f3_fields(c); a.pack = c->s_pack;
  a.kx2 = c->k2n[0]; a.ky2 = c->k2n[1]; a.kz2 = c->k2n[2];
  a.invM = c->L.invM; a.dV = c->dV; a.kappa = kappa;
  a.spec0 = c->s_spec0; a.spec1 = c->s_spec1; a.X = c->s_X; a.out = out; a.cpart = cpart; a.part = c->s_part;
  a.eps_out = mode == F3_APPLY ? nullptr : c->eps + n0;
  a.use_shift = c->f.subtract_mean_energy; a.normalize = c->f.normalize; a.do_dens = do_dens;
  a.cpref = c->cpref + n0; a.w_a = c->w_a + n0; a.w_b = c->w_b + n0; a.acc = c->s_acc; a.sync = c->s_sync;
  a.n = (int)n; a.G = (int)(2 * n);
  cudaMemsetAsync(c->s_sync, 0, sizeof(F3Sync) + (size_t)5 * a.G * sizeof(int), st);
  LAUNCH(c, k_f3_pack, nb(P.M, 256), 256, 0, st, a.F, 1, P.M, c->s_pack);
  const double M = (double)P.M;
  WORK(c, M * n * (mode == F3_CORR ? 96.0 : 64.0), 5.0 * M * 18.0 * 2.0 * 2 * 2 * n);
  const char* name = mode == F3_APPLY ? "k_f6_mega_apply" : mode == F3_CORR ? "k_f6_mega_corr" : "k_f6_mega_rhs";
  {
    const int IT = F6_N / 2 + F6_N / 2 + F6_N + (mode == F3_APPLY ? 0 : F6_ND);
    const long total = (long)(a.G + 4) * IT;
    const int grid = (int)(total < 148 ? total : 148);
    void (*k)(F6Mega) = mode == F3_APPLY ? k_f6_mega<F3_APPLY> : mode == F3_CORR ? k_f6_mega<F3_CORR> : k_f6_mega<F3_RHS>;
    LAUNCHN(c, name, k, grid, F6_THREADS, 2 * F6_TILE * 16, st, a);
    if (c->err_host) cudaMemcpyAsync(c->err_host, &c->s_sync->error, sizeof(int), cudaMemcpyDeviceToHost, st);
  }
}

static void f3_scal(wslda_ctx* c, int q, cudaStream_t st, int64_t n0, int cnt, int mode, int use_shift, double kappa,
                    double* eps_user) {
  F3Scal s;
  s.part = c->f_part[q]; s.cnt = cnt; s.NX = c->P.N[0]; s.mode = mode; s.use_shift = use_shift; s.normalize = c->f.normalize;
  s.dV = c->dV; s.kappa = kappa; s.eps = c->eps + n0; s.eps_user = eps_user; s.scale_new = c->scale2 + n0;
  LAUNCH(c, k_f3_scal, (cnt + 3) / 4, 128, 0, st, s);
}

static wslda_status f3_apply_h(wslda_ctx* c, const cplx* psi, cplx* hpsi, double* eps_dev, int64_t n_first, int64_t n_count,
                               cudaStream_t st) {
  const int64_t M = c->P.M;
  if (c->P.f6) {
    if (n_count > 0) {
      f6_mega(c, st, F3_APPLY, psi + 2 * n_first * M, nullptr, n_first, n_count, hpsi + 2 * n_first * M, nullptr, 0.0, 0);
      LAUNCH(c, k_f6_scal, (unsigned)((n_count + 3) / 4), 128, 0, st, c->s_part, (int)n_count, c->dV, c->eps + n_first,
             eps_dev ? eps_dev + n_first : (double*)nullptr);
    }
    return cuda_check(c, "apply_h");
  }
  if (c->P.mega && n_count > 0 && f3_uses_t3(c)) {           // eps_n comes out of the stage kernel itself
    f3_mega(c, st, F3_APPLY, psi + 2 * n_first * M, nullptr, n_first, n_count, hpsi + 2 * n_first * M, nullptr, 0.0, 0,
            eps_dev ? eps_dev + n_first : nullptr);
    return cuda_check(c, "apply_h");
  }
  if (c->P.mega && n_count > 0) {
    f3_mega(c, st, F3_APPLY, psi + 2 * n_first * M, nullptr, n_first, n_count, hpsi + 2 * n_first * M, nullptr, 0.0, 0);
    F3Scal s;
    s.part = c->m_part; s.cnt = (int)n_count; s.NX = c->P.N[0]; s.mode = F3_APPLY; s.use_shift = 1; s.normalize = 0;
    s.dV = c->dV; s.kappa = 0.0; s.eps = c->eps + n_first; s.eps_user = eps_dev ? eps_dev + n_first : nullptr; s.scale_new = nullptr;
    LAUNCH(c, k_f3_scal, (unsigned)((n_count + 3) / 4), 128, 0, st, s);
    return cuda_check(c, "apply_h");
  }
  for (int64_t n0 = n_first; n0 < n_first + n_count; n0 += c->P.fc) {
    const int cnt = (int)((n_first + n_count - n0 < c->P.fc) ? n_first + n_count - n0 : c->P.fc);
    f3_hpsi(c, 0, st, psi + 2 * n0 * M, nullptr, n0, cnt, F3_APPLY, hpsi + 2 * n0 * M, nullptr, 0.0);
    f3_scal(c, 0, st, n0, cnt, F3_APPLY, 1, 0.0, eps_dev ? eps_dev + n0 : nullptr);
  }
  return cuda_check(c, "apply_h");
}

// ---- the Alg. 2 step -----------------------------------------------------------------------------------------
struct F3Step {
  cplx* phi; HistPtrs h; cplx* cpart; AbmCoef k; double c0dt;
  cudaStream_t user;
};

static inline cudaStream_t f3_stream(wslda_ctx* c, const F3Step& s, int q) { return c->P.ns > 1 ? c->aux[q] : s.user; }
static void f3_fork(wslda_ctx* c, const F3Step& s) {
  if (c->P.ns == 1) return;
  cudaEventRecord(c->ev_fork, s.user);
  for (int q = 0; q < c->P.ns; ++q) cudaStreamWaitEvent(c->aux[q], c->ev_fork, 0);
}
static void f3_join(wslda_ctx* c, const F3Step& s) {
  if (c->P.ns == 1) return;
  for (int q = 0; q < c->P.ns; ++q) { cudaEventRecord(c->ev_join[q], c->aux[q]); cudaStreamWaitEvent(s.user, c->ev_join[q], 0); }
}

static F3Dens f3_dens_args(wslda_ctx* c, int q, int64_t n0, int first) {
  F3Dens d; d.cpref = c->cpref + n0; d.w_a = c->w_a + n0; d.w_b = c->w_b + n0; d.acc = c->f_acc[q]; d.first = first;
  return d;
}

// Alg. 2 step 1-2: predictor P -> phi buffer, C_part -> oldest history buffer, scale_n = 1/|P|
static void f3_stage1(wslda_ctx* c, const F3Step& s, int q, cudaStream_t st, int64_t n0, int cnt) {
  const Plan& P = c->P;
  const int64_t off = 2 * n0 * P.M;
  HistPtrs h = s.h;
  for (int j = 0; j < 5; ++j) if (h.f[j]) h.f[j] += off;
  WORK(c, 32.0 * P.M * cnt * (1 + c->m + 2), 0);
  LAUNCH(c, k_f3_combine, dim3(P.nblk, (unsigned)cnt), P.pt_threads, 0, st, s.phi + off, h, s.cpart + off, s.k, P.M,
         c->f.normalize ? c->f_partn[q] : (double*)nullptr, P.nblk, c->f_cnt[q], c->dV, c->scale + n0);
}
// Alg. 2 steps 3-4, 8: phi_new = C_part + c0 dt f(P), normalised, written over P (+ its densities)
static void f3_stage2(wslda_ctx* c, const F3Step& s, int q, cudaStream_t st, int64_t n0, int cnt, int do_dens, int first) {
  const Plan& P = c->P;
  const int64_t off = 2 * n0 * P.M;
  const double* sc = c->f.normalize ? c->scale + n0 : nullptr;
  f3_hpsi(c, q, st, s.phi + off, sc, n0, cnt, F3_CORR, c->f_X[q], s.cpart + off, s.c0dt);
  f3_scal(c, q, st, n0, cnt, F3_CORR, c->f.subtract_mean_energy, s.c0dt, nullptr);
  F3Fin2 f;
  f.X = c->f_X[q]; f.phi = s.phi + off; f.scaleP = sc; f.eps = c->eps + n0; f.scale_new = c->scale2 + n0; f.kappa = s.c0dt;
  f.cnt = cnt; f.M = P.M; f.do_dens = do_dens; f.d = f3_dens_args(c, q, n0, first);
  WORK(c, 32.0 * P.M * cnt, 0);                            // writes phi_new
  LAUNCH(c, k_f3_fin2, nb(P.M, 128), 128, 0, st, f);
}
// Alg. 2 step 9: f(phi_new) -> the recycled oldest history buffer
static void f3_stage3(wslda_ctx* c, const F3Step& s, int q, cudaStream_t st, int64_t n0, int cnt) {
  const Plan& P = c->P;
  const int64_t off = 2 * n0 * P.M;
  f3_hpsi(c, q, st, s.phi + off, nullptr, n0, cnt, F3_RHS, c->f_X[q], nullptr, 0.0);
  f3_scal(c, q, st, n0, cnt, F3_RHS, c->f.subtract_mean_energy, 0.0, nullptr);
  WORK(c, 32.0 * P.M * cnt, 0);                            // writes f_new
  LAUNCH(c, k_f3_fin3, dim3(nb(2 * P.M, 256), (unsigned)cnt), 256, 0, st, c->f_X[q], s.phi + off, c->eps + n0, s.cpart + off, 2 * P.M);
}

static void potentials(wslda_ctx* c, cudaStream_t st, bool fresh = true);
static unsigned step_mask(const wslda_ctx* c);

static void f3_dens_final(wslda_ctx* c, int used, cudaStream_t st) {
  const int64_t M = c->P.M;
  LAUNCH(c, k_f3_dens_final, nb(4 * M, 256), 256, 0, st, c->f_acc[0], used, (int64_t)(c->P.fast_stream_bytes / 8), M, c->raw);
}

// The fused step serves functionals that consume rho and nu only, and -- on cubic 32^3 lattices with the persistent
// kernels -- tau and j as well (polarised ASLDA; A_sigma = (1 - alpha_sigma) j_sigma / rho_sigma): the gradient densities are
// then taken axis by axis (gdens.cuh) after each stage.
static bool f3_step_ok(const wslda_ctx* c) {
  if (!c->P.fast) return false;
  if (c->f.func_id == WSLDA_FUNC_FIXED) return true;
  const unsigned m = step_mask(c);
  if (m == (WSLDA_D_RHO | WSLDA_D_NU)) return true;
  return !(m & ~(WSLDA_D_RHO | WSLDA_D_NU | WSLDA_D_TAU | WSLDA_D_J | WSLDA_D_BP)) && c->P.mega && gdens_ok(c);
}

static void f3_abm_step(wslda_ctx* c, const F3Step& s) {
  const Plan& P = c->P;
  const int64_t n_wf = P.n_wf;
  const int fc = P.fc, ns = P.ns;
  const int64_t n_chunks = (n_wf + fc - 1) / fc;
  const int used = (int)(n_chunks < ns ? n_chunks : ns);
  auto cnt_of = [&](int64_t k) { return (int)((n_wf - k * fc < fc) ? n_wf - k * fc : fc); };
  const bool fixed = c->f.func_id == WSLDA_FUNC_FIXED;
  if (P.mega) {                                // stage 1 in chunks, stages 2 and 3 as persistent dataflow kernels
    f3_fork(c, s);
    for (int64_t k = 0; k < n_chunks; ++k) {
      const int q = (int)(k % ns); cudaStream_t st = f3_stream(c, s, q);
      const int64_t n0 = k * fc; const int cnt = cnt_of(k);
      f3_stage1(c, s, q, st, n0, cnt);
      if (!fixed) {
        F3DensOnly d;
        d.psi = s.phi + 2 * n0 * P.M; d.scale = c->f.normalize ? c->scale + n0 : nullptr; d.cnt = cnt; d.M = P.M;
        d.d = f3_dens_args(c, q, n0, k < ns);
        WORK(c, 0, 0);
        LAUNCH(c, k_f3_dens, nb(P.M, 64), 256, 0, st, d);
      }
    }
    f3_join(c, s);
    const unsigned gm = fixed ? 0u : step_mask(c) & (WSLDA_D_TAU | WSLDA_D_J);      // gradient densities the functional consumes
    if (!fixed) {
      f3_dens_final(c, used, s.user);
      if (gm) gdens(c, s.phi, 0, n_wf, gm, 0, s.user, c->f.normalize ? c->scale : nullptr);     // of the (unnormalised) predictor
      if (step_mask(c) & WSLDA_D_BP) gdens_bp(c, s.phi, 0, n_wf, 0, s.user, c->f.normalize ? c->scale : nullptr);
      potentials(c, s.user);
    }
    f3_mega(c, s.user, F3_CORR, s.phi, c->f.normalize ? c->scale : nullptr, 0, n_wf, s.phi, s.cpart, s.c0dt, !fixed);
    if (!fixed) {
      const int64_t mG = f3_uses_t3(c) ? (n_wf + c->t3_gs - 1) / c->t3_gs : c->P.mG;
      const int slots = (int)(mG < F3_RING ? mG : F3_RING);
      LAUNCH(c, k_f3_dens_final, nb(4 * P.M, 256), 256, 0, s.user, c->m_acc, slots, (int64_t)(4 * P.M), P.M, c->raw);
      if (gm) gdens(c, s.phi, 0, n_wf, gm, 0, s.user);                  // of phi_new (normalised)
      if (step_mask(c) & WSLDA_D_BP) gdens_bp(c, s.phi, 0, n_wf, 0, s.user);
      potentials(c, s.user);
    }
    f3_mega(c, s.user, F3_RHS, s.phi, nullptr, 0, n_wf, s.cpart, nullptr, 0.0, 0);
    return;
  }
  f3_fork(c, s);
  if (fixed) {
    for (int64_t k = 0; k < n_chunks; ++k) {
      const int q = (int)(k % ns); cudaStream_t st = f3_stream(c, s, q);
      f3_stage1(c, s, q, st, k * fc, cnt_of(k));
      f3_stage2(c, s, q, st, k * fc, cnt_of(k), 0, 0);
      f3_stage3(c, s, q, st, k * fc, cnt_of(k));
    }
    f3_join(c, s);
    return;
  }
  for (int64_t k = 0; k < n_chunks; ++k) {
    const int q = (int)(k % ns); cudaStream_t st = f3_stream(c, s, q);
    const int64_t n0 = k * fc; const int cnt = cnt_of(k);
    f3_stage1(c, s, q, st, n0, cnt);
    F3DensOnly d;
    d.psi = s.phi + 2 * n0 * P.M; d.scale = c->f.normalize ? c->scale + n0 : nullptr; d.cnt = cnt; d.M = P.M;
    d.d = f3_dens_args(c, q, n0, k < ns);
    LAUNCH(c, k_f3_dens, nb(P.M, 64), 256, 0, st, d);
  }
  f3_join(c, s);
  f3_dens_final(c, used, s.user);
  potentials(c, s.user);
  f3_fork(c, s);
  for (int64_t k = 0; k < n_chunks; ++k) {
    const int q = (int)(k % ns);
    f3_stage2(c, s, q, f3_stream(c, s, q), k * fc, cnt_of(k), 1, k < ns);
  }
  f3_join(c, s);
  f3_dens_final(c, used, s.user);
  potentials(c, s.user);
  f3_fork(c, s);
  for (int64_t k = 0; k < n_chunks; ++k) {
    const int q = (int)(k % ns);
    f3_stage3(c, s, q, f3_stream(c, s, q), k * fc, cnt_of(k));
  }
  f3_join(c, s);
}
