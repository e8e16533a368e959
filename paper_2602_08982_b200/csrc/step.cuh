// step.cuh -- time stepping: right-hand side, Taylor starter (Eqs. 52-54) and the
// Adams-Bashforth-Moulton predictor-corrector following Alg. 2.  General chunked path:
// spinors are processed in chunks whose intermediates (spectral terms, H psi) stay in L2-sized scratch.
#pragma once
#include "fast_step.cuh"

// Eqs. 46-50
static const double AB3[5] = {23.0 / 12, -16.0 / 12, 5.0 / 12, 0, 0};
static const double AB4[5] = {55.0 / 24, -59.0 / 24, 37.0 / 24, -9.0 / 24, 0};
static const double AB5[5] = {1901.0 / 720, -2774.0 / 720, 2616.0 / 720, -1274.0 / 720, 251.0 / 720};
static const double AM4[5] = {9.0 / 24, 19.0 / 24, -5.0 / 24, 1.0 / 24, 0};
static const double AM5[5] = {251.0 / 720, 646.0 / 720, -264.0 / 720, 106.0 / 720, -19.0 / 720};

// densities the functional consumes inside a step: rho and nu always; tau only where alpha depends on the
// polarisation (ASLDA without force_a1) and the densities are not spin-folded (then p = 0 and the tau term
// of V_sigma cancels exactly).
static unsigned step_mask(const wslda_ctx* c) {
  unsigned m = WSLDA_D_RHO | WSLDA_D_NU;
  if (c->f.func_id == WSLDA_FUNC_ASLDA && !c->f.force_a1 && !c->f.spin_symmetric) m |= WSLDA_D_TAU;
  if (c->f.current_terms && c->f.func_id == WSLDA_FUNC_ASLDA && !c->f.force_a1) m |= WSLDA_D_J;     // A_sigma follows j
  if (c->f.quantum_friction) m |= WSLDA_D_J | WSLDA_D_BP;                                          // div j (Eq. 66), B' (Eq. 68)
  return m;
}
static inline int64_t chunk_len(const wslda_ctx* c, int64_t n0) {
  return (c->P.n_wf - n0 < c->P.chunk_n) ? c->P.n_wf - n0 : c->P.chunk_n;
}

// densities of a whole buffer (optionally scaled per spinor) followed by the potential update
static void rebuild(wslda_ctx* c, const cplx* psi, const double* scale, cudaStream_t st) {
  if (c->f.func_id == WSLDA_FUNC_FIXED) return;
  const int64_t M = c->P.M;
  for (int64_t n0 = 0; n0 < c->P.n_wf; n0 += c->P.chunk_n)
    dens_chunk(c, psi + 2 * n0 * M, scale ? scale + n0 : nullptr, n0, chunk_len(c, n0), step_mask(c), n0 > 0, st);
  potentials(c, st);
}

// eps_n of the chunk from the partials of the last h_chunk (null when the shift of Eq. 44 is off)
static const double* eps_chunk(wslda_ctx* c, int64_t n0, int64_t cnt, cudaStream_t st) {
  if (!c->f.subtract_mean_energy) return nullptr;
  LAUNCH(c, k_from_partials, nb(cnt * 32, 128), 128, 0, st, c->part_e, c->P.nblk, cnt, c->dV, 0, c->eps + n0, (double*)nullptr);
  return c->eps + n0;
}
static void scale_chunk_from_partials(wslda_ctx* c, int64_t n0, int64_t cnt, cudaStream_t st) {
  LAUNCH(c, k_from_partials, nb(cnt * 32, 128), 128, 0, st, c->part_n, c->P.nblk, cnt, c->dV, 1, c->scale + n0, (double*)nullptr);
}

// f = -i (H - eps) psi for the chunk; psi_chunk in the caller's buffer, scaled on the fly; the scaled state is
// written back when write_back is set.
static void rhs_chunk(wslda_ctx* c, cplx* psi_chunk, const double* scale_chunk, int64_t n0, int64_t cnt, cplx* f_chunk,
                      int write_back, cudaStream_t st) {
  const Plan& P = c->P;
  h_chunk(c, psi_chunk, scale_chunk, n0, cnt, c->scr[4], c->f.subtract_mean_energy != 0, st);
  const double* eps = eps_chunk(c, n0, cnt, st);
  WORK(c, 64.0 * P.M * cnt, 0);    // reads psi (H psi is scratch), writes f
  LAUNCH(c, k_rhs, dim3(P.nblk, (unsigned)cnt), P.pt_threads, 0, st, psi_chunk, scale_chunk, c->scr[4], eps, 0, write_back,
         f_chunk, (const cplx*)nullptr, 0.0, P.M, (double*)nullptr, P.nblk);
}

// Eqs. 53/54 for one chunk: scr[6] = sum_{k<=r} (-i s)^k / k! G^k phi, G = H - eps_n with the current
// potentials and eps_n fixed at its value for phi.  Uses scr[4] (H t), scr[5] (t), scr[6] (result).
static void taylor_chunk(wslda_ctx* c, const cplx* phi_chunk, int64_t n0, int64_t cnt, double s, int r, cudaStream_t st) {
  const Plan& P = c->P;
  const int64_t tot = 2 * cnt * P.M;
  LAUNCH(c, k_copy2, nb(tot, 256), 256, 0, st, phi_chunk, c->scr[5], c->scr[6], tot);
  const double* eps = nullptr;
  cplx coef = make_double2(1.0, 0.0);
  for (int k = 1; k <= r; ++k) {
    h_chunk(c, c->scr[5], nullptr, n0, cnt, c->scr[4], k == 1 && c->f.subtract_mean_energy, st);
    if (k == 1) eps = eps_chunk(c, n0, cnt, st);
    coef = cmul(coef, make_double2(0.0, -s / (double)k));
    LAUNCH(c, k_taylor_acc, dim3(P.nblk, (unsigned)cnt), P.pt_threads, 0, st, c->scr[5], c->scr[4], eps, coef, c->scr[6], P.M);
  }
}

static void rotate_history(void** f_hist, int m) {      // Alg. 2 steps 5-7: the oldest buffer becomes slot 0
  void* last = f_hist[m - 1];
  for (int i = m - 1; i > 0; --i) f_hist[i] = f_hist[i - 1];
  f_hist[0] = last;
}

static wslda_status check_hist(wslda_ctx* c, void* phi, void** f_hist) {
  if (!c) return WSLDA_EINVAL;
  if (!phi || !f_hist) return fail(c, WSLDA_EINVAL, "abm: null buffer");
  for (int i = 0; i < c->m; ++i) {
    if (!f_hist[i] || f_hist[i] == phi) return fail(c, WSLDA_EINVAL, "abm: history buffers must be distinct non-null device buffers");
    for (int j = 0; j < i; ++j) if (f_hist[i] == f_hist[j]) return fail(c, WSLDA_EINVAL, "abm: history buffers must be distinct");
  }
  return WSLDA_OK;
}

extern "C" wslda_status wslda_abm_init(wslda_ctx* c, void* phi_, void** f_hist, double dt, int selfstart, void* stream) {
  wslda_status rc = check_hist(c, phi_, f_hist);
  if (rc) return rc;
  const Plan& P = c->P;
  const int64_t M = P.M, n_wf = P.n_wf;
  const int m = c->m;
  cplx* phi = (cplx*)phi_;
  cudaStream_t st = S(stream);
  if (!selfstart) {                                      // stationary start: f_k = 0
    for (int i = 0; i < m; ++i) cudaMemsetAsync(f_hist[i], 0, (size_t)n_wf * 2 * M * 16, st);
    rebuild(c, phi, nullptr, st);
    return cuda_check(c, "abm_init");
  }
  const int r = c->f.am_order;                           // truncation order = corrector order
  const bool fixed = c->f.func_id == WSLDA_FUNC_FIXED;
  rebuild(c, phi, nullptr, st);
  for (int64_t n0 = 0; n0 < n_wf; n0 += P.chunk_n)
    rhs_chunk(c, phi + 2 * n0 * M, nullptr, n0, chunk_len(c, n0), (cplx*)f_hist[0] + 2 * n0 * M, 0, st);
  for (int s = 1; s < m; ++s) {
    if (!fixed) {                                        // Eq. 53: midpoint predictor, only its densities are needed
      for (int64_t n0 = 0; n0 < n_wf; n0 += P.chunk_n) {
        const int64_t cnt = chunk_len(c, n0);
        taylor_chunk(c, phi + 2 * n0 * M, n0, cnt, 0.5 * dt, r, st);
        dens_chunk(c, c->scr[6], nullptr, n0, cnt, step_mask(c), n0 > 0, st);
      }
      potentials(c, st);                                 // H(phi^(p), t + dt/2)
    }
    for (int64_t n0 = 0; n0 < n_wf; n0 += P.chunk_n) {   // Eq. 54
      const int64_t cnt = chunk_len(c, n0);
      taylor_chunk(c, phi + 2 * n0 * M, n0, cnt, dt, r, st);
      if (c->f.normalize) {
        LAUNCH(c, k_norm_partials, dim3(P.nblk, (unsigned)cnt), P.pt_threads, 0, st, c->scr[6], M, c->part_n, P.nblk);
        scale_chunk_from_partials(c, n0, cnt, st);
        LAUNCH(c, k_scale_spinors, dim3(P.nblk, (unsigned)cnt), P.pt_threads, 0, st, c->scr[6], c->scale + n0, M);
      }
      cudaMemcpyAsync(phi + 2 * n0 * M, c->scr[6], (size_t)cnt * 2 * M * 16, cudaMemcpyDeviceToDevice, st);
    }
    rotate_history(f_hist, m);
    rebuild(c, phi, nullptr, st);
    for (int64_t n0 = 0; n0 < n_wf; n0 += P.chunk_n)
      rhs_chunk(c, phi + 2 * n0 * M, nullptr, n0, chunk_len(c, n0), (cplx*)f_hist[0] + 2 * n0 * M, 0, st);
  }
  return cuda_check(c, "abm_init");
}

struct StepBufs { cplx* phi; HistPtrs h; cplx* cpart; AbmCoef k; double c0dt; };

// Alg. 2 step 1 (+2): predictor and partial corrector for one chunk; the norm of P goes to scale[]
static void stage1(wslda_ctx* c, const StepBufs& b, int64_t n0, int64_t cnt, cudaStream_t st) {
  const Plan& P = c->P;
  const int64_t off = 2 * n0 * P.M;
  HistPtrs h = b.h;
  for (int j = 0; j < 5; ++j) if (h.f[j]) h.f[j] += off;
  WORK(c, 32.0 * P.M * cnt * (1 + c->m + 2), 0);   // reads phi, f_1..f_m; writes P, C_part
  LAUNCH(c, k_abm_combine, dim3(P.nblk, (unsigned)cnt), P.pt_threads, 0, st, b.phi + off, h, b.cpart + off, b.k, P.M,
         c->f.normalize ? c->part_n : (double*)nullptr, P.nblk);
  if (c->f.normalize) scale_chunk_from_partials(c, n0, cnt, st);
}
// Alg. 2 steps 3-4 (+8): f(P), phi_new = C_part + c0 dt f(P) in place over P; its norm goes to scale[]
static void stage2(wslda_ctx* c, const StepBufs& b, int64_t n0, int64_t cnt, cudaStream_t st) {
  const Plan& P = c->P;
  const int64_t off = 2 * n0 * P.M;
  const double* sc = c->f.normalize ? c->scale + n0 : nullptr;
  h_chunk(c, b.phi + off, sc, n0, cnt, c->scr[4], c->f.subtract_mean_energy != 0, st);
  const double* eps = eps_chunk(c, n0, cnt, st);
  WORK(c, 96.0 * P.M * cnt, 0);    // reads P, C_part; writes phi_new
  LAUNCH(c, k_rhs, dim3(P.nblk, (unsigned)cnt), P.pt_threads, 0, st, b.phi + off, sc, c->scr[4], eps, 1, 0, (cplx*)nullptr,
         b.cpart + off, b.c0dt, P.M, c->f.normalize ? c->part_n : (double*)nullptr, P.nblk);
  if (c->f.normalize) scale_chunk_from_partials(c, n0, cnt, st);
}
// Alg. 2 step 9: f(phi_new) into the recycled oldest history buffer; phi_new is stored normalised
static void stage3(wslda_ctx* c, const StepBufs& b, int64_t n0, int64_t cnt, cudaStream_t st) {
  const int64_t off = 2 * n0 * c->P.M;
  const double* sc = c->f.normalize ? c->scale + n0 : nullptr;
  rhs_chunk(c, b.phi + off, sc, n0, cnt, b.cpart + off, c->f.normalize, st);
}

extern "C" wslda_status wslda_abm_step(wslda_ctx* c, void* phi_, void** f_hist, double dt, void* stream) {
  wslda_status rc = check_hist(c, phi_, f_hist);
  if (rc) return rc;
  const Plan& P = c->P;
  const int64_t M = P.M, n_wf = P.n_wf;
  const int m = c->m, ab = c->f.ab_order, am = c->f.am_order;
  cudaStream_t st = S(stream);
  const double* B = ab == 3 ? AB3 : ab == 4 ? AB4 : AB5;
  const double* C = am == 4 ? AM4 : AM5;
  StepBufs b;
  b.phi = (cplx*)phi_;
  for (int j = 0; j < 5; ++j) { b.h.f[j] = j < m ? (const cplx*)f_hist[j] : nullptr; b.k.b[j] = B[j] * dt; b.k.c[j] = C[j] * dt; }
  b.k.ab = ab; b.k.am = am;
  b.cpart = (cplx*)f_hist[m - 1];
  b.c0dt = C[0] * dt;
  const bool fixed = c->f.func_id == WSLDA_FUNC_FIXED;
  const unsigned mask = step_mask(c);
  if (c->P.oc && (fixed || mask == (WSLDA_D_RHO | WSLDA_D_NU))) {   // fused on-chip stages (onchip_step.cuh)
    oc_pred(c, st, b.phi, b.h, b.cpart, b.k, !fixed);       // the predictor is stored normalised: no scale afterwards
    if (!fixed) potentials(c, st);
    oc_launch(c, st, OC_CORR, b.phi, nullptr, 0, n_wf, b.phi, b.cpart, b.c0dt, !fixed, c->eps);
    if (!fixed) potentials(c, st);
    oc_launch(c, st, OC_RHS, b.phi, nullptr, 0, n_wf, b.cpart, nullptr, 0.0, 0, c->eps);
  } else if (c->P.f6 && (fixed || mask == (WSLDA_D_RHO | WSLDA_D_NU) ||
                         (!(mask & ~(WSLDA_D_RHO | WSLDA_D_NU | WSLDA_D_TAU | WSLDA_D_J | WSLDA_D_BP)) && gdens_ok(c)))) {   // 64^3 persistent kernels (mega64.cuh)
    // (polarised ASLDA, quantum friction: tau, j, B' by the axis-by-axis density kernels after each stage, as on the 32^3 path)
    const unsigned gm = fixed ? 0u : mask & (WSLDA_D_TAU | WSLDA_D_J), pm = mask & (WSLDA_D_RHO | WSLDA_D_NU);
    const bool bp = !fixed && (mask & WSLDA_D_BP);
    const double* scg = c->f.normalize ? c->scale : nullptr;
    if (fixed) {                                         // no density barrier: one predictor launch over the whole batch
      WORK(c, 32.0 * M * n_wf * (1 + c->m + 2), 0);
      LAUNCH(c, k_abm_combine, dim3(P.nblk, (unsigned)n_wf), P.pt_threads, 0, st, b.phi, b.h, b.cpart, b.k, M,
             c->f.normalize ? c->s_partn : (double*)nullptr, P.nblk);
      if (c->f.normalize)
        LAUNCH(c, k_from_partials, nb(n_wf * 32, 128), 128, 0, st, c->s_partn, P.nblk, n_wf, c->dV, 1, c->scale, (double*)nullptr);
    } else {
      for (int64_t n0 = 0; n0 < n_wf; n0 += P.chunk_n) {
        const int64_t cnt = chunk_len(c, n0);
        stage1(c, b, n0, cnt, st);
        dens_chunk(c, b.phi + 2 * n0 * M, scg ? scg + n0 : nullptr, n0, cnt, pm, n0 > 0, st);
      }
      if (gm) gdens(c, b.phi, 0, n_wf, gm, 0, st, scg);
      if (bp) gdens_bp(c, b.phi, 0, n_wf, 0, st, scg);
      potentials(c, st);
    }
    f6_mega(c, st, F3_CORR, b.phi, scg, 0, n_wf, b.phi, b.cpart, b.c0dt, !fixed);
    if (!fixed) {
      const int slots = (int)(n_wf < F6_RING ? n_wf : F6_RING);
      LAUNCH(c, k_f3_dens_final, nb(4 * M, 256), 256, 0, st, c->s_acc, slots, (int64_t)(4 * M), M, c->raw);
      if (gm) gdens(c, b.phi, 0, n_wf, gm, 0, st);
      if (bp) gdens_bp(c, b.phi, 0, n_wf, 0, st);
      potentials(c, st);
    }
    f6_mega(c, st, F3_RHS, b.phi, nullptr, 0, n_wf, b.cpart, nullptr, 0.0, 0);
  } else if (f3_step_ok(c)) {                            // fused 3-D path (fast_step.cuh)
    F3Step s; s.phi = b.phi; s.h = b.h; s.cpart = b.cpart; s.k = b.k; s.c0dt = b.c0dt; s.user = st;
    f3_abm_step(c, s);
  } else if (fixed) {                                    // no global barrier: run the three stages chunk by chunk
    for (int64_t n0 = 0; n0 < n_wf; n0 += P.chunk_n) {
      const int64_t cnt = chunk_len(c, n0);
      stage1(c, b, n0, cnt, st); stage2(c, b, n0, cnt, st); stage3(c, b, n0, cnt, st);
    }
  } else {
    const double* scg = c->f.normalize ? c->scale : nullptr;
    for (int64_t n0 = 0; n0 < n_wf; n0 += P.chunk_n) {
      const int64_t cnt = chunk_len(c, n0);
      stage1(c, b, n0, cnt, st);
      dens_chunk(c, b.phi + 2 * n0 * M, scg ? scg + n0 : nullptr, n0, cnt, mask, n0 > 0, st);
    }
    potentials(c, st);
    for (int64_t n0 = 0; n0 < n_wf; n0 += P.chunk_n) {
      const int64_t cnt = chunk_len(c, n0);
      stage2(c, b, n0, cnt, st);
      dens_chunk(c, b.phi + 2 * n0 * M, scg ? scg + n0 : nullptr, n0, cnt, mask, n0 > 0, st);
    }
    potentials(c, st);
    for (int64_t n0 = 0; n0 < n_wf; n0 += P.chunk_n) stage3(c, b, n0, chunk_len(c, n0), st);
  }
  rotate_history(f_hist, m);
  return cuda_check(c, "abm_step");
}

extern "C" wslda_status wslda_abm_step_host(wslda_ctx* c, void* phi_host, void** f_hist_host, void* phi_dev,
                                            void** f_hist_dev, double dt, void* stream) {
  if (!c || !phi_host || !f_hist_host) return fail(c, WSLDA_EINVAL, "abm_step_host: null host buffer");
  wslda_status rc = check_hist(c, phi_dev, f_hist_dev);
  if (rc) return rc;
  cudaStream_t st = S(stream);
  const size_t bytes = (size_t)c->P.n_wf * 2 * c->P.M * 16;
  cudaMemcpyAsync(phi_dev, phi_host, bytes, cudaMemcpyHostToDevice, st);
  for (int i = 0; i < c->m; ++i) {
    if (!f_hist_host[i]) return fail(c, WSLDA_EINVAL, "abm_step_host: null host history buffer");
    cudaMemcpyAsync(f_hist_dev[i], f_hist_host[i], bytes, cudaMemcpyHostToDevice, st);
  }
  rc = wslda_abm_step(c, phi_dev, f_hist_dev, dt, stream);
  if (rc) return rc;
  rotate_history(f_hist_host, c->m);
  cudaMemcpyAsync(phi_host, phi_dev, bytes, cudaMemcpyDeviceToHost, st);
  cudaMemcpyAsync(f_hist_host[0], f_hist_dev[0], bytes, cudaMemcpyDeviceToHost, st);
  cudaStreamSynchronize(st);
  return cuda_check(c, "abm_step_host");
}
