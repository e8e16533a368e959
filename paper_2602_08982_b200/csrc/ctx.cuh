// ctx.cuh -- context object, workspace plan, creation and the setters (host side of libwslda).
#pragma once
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <vector>
#include <algorithm>
#include <utility>
#include "density.cuh"
#include "fft_large.cuh"
#include "fast3d.cuh"
#include "mega3d.cuh"
#include "mega3s.cuh"
#include "mega3t.cuh"
#include "mega3m.cuh"
#include "mega64.cuh"
#include "gdens.cuh"
#include "kernels.cuh"

struct Plan {
  int nd, N[3], lg[3];
  int64_t M, n_wf, chunk_n;
  int nblk, pt_threads;         // pointwise kernels: blocks per spinor, threads per block
  bool onchip; int G;           // whole-lattice-in-shared-memory regime, components per CTA
  int PX, lgT;                  // large regime: x-planes per CTA, log2 of the x-line tile width
  int dG;                       // max density groups per chunk
  int nscr;
  // fused 3-D path (fast3d.cuh): enabled flag, spinors per chunk, concurrent streams, per-stream scratch
  int fast, fc, ns;
  size_t off_fast, fast_spec_bytes, fast_part_bytes, fast_stream_bytes;
  // persistent dataflow kernels (mega3d.cuh): enabled flag, spinors per group, number of groups, ring buffers
  // fused on-chip stages (onchip_step.cuh): enabled flag, spinors per CTA batch, persistent grid, density partials
  int oc, ocS, oc_grid;
  size_t off_oc, oc_dpart_bytes;
  // 64^3 persistent kernels (mega64.cuh)
  int f6;
  size_t off_f6, f6_ring_bytes, f6_part_bytes, f6_acc_bytes, f6_sync_bytes, f6_pack_bytes, f6_partn_bytes;
  int mega, gs, mG, sep;
  size_t off_mega, mega_ring_bytes, mega_part_bytes, mega_acc_bytes, mega_sync_bytes, mega_pack_bytes;
  size_t off_cur, off_obs, off_qf;
  size_t off_tables, off_perwf, off_fields, off_part, off_dpart, off_scr, scr_bytes, total;
};

// process-wide tuning (wslda_set_tuning); all zeros = the library's defaults
static wslda_tuning g_tune = {};
extern "C" wslda_status wslda_set_tuning(const wslda_tuning* t) {
  if (t) g_tune = *t; else g_tune = wslda_tuning{};
  return WSLDA_OK;
}

static int ilog2(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }
static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// status: 0 ok, else a wslda_status
static int make_plan(const int dims[3], int mode, int64_t n_wf, const wslda_functional* f, Plan& P) {
  if (!dims || !f || mode < 1 || mode > 3 || n_wf < 1) return WSLDA_EINVAL;
  for (int d = 0; d < 3; ++d) if (dims[d] < 1) return WSLDA_EINVAL;
  bool okpair = (f->ab_order == 3 && f->am_order == 4) || (f->ab_order == 4 && f->am_order == 4) ||
                (f->ab_order == 4 && f->am_order == 5) || (f->ab_order == 5 && f->am_order == 5);
  if (!okpair || f->kin_form < 0 || f->kin_form > 2 || f->func_id < 0 || f->func_id > 2) return WSLDA_EINVAL;
  if (f->quantum_friction && (f->func_id == WSLDA_FUNC_FIXED || !(f->qf_rho0 > 0) || !(f->qf_nreq > 0))) return WSLDA_EINVAL;
  P.nd = mode; P.M = 1;
  for (int d = 0; d < 3; ++d) {
    P.N[d] = d < mode ? dims[d] : 1;
    if (d < mode && (dims[d] < 2 || (dims[d] & (dims[d] - 1)))) return WSLDA_EUNSUPPORTED;
    P.lg[d] = ilog2(P.N[d]);
    P.M *= P.N[d];
  }
  P.n_wf = n_wf;
  const int64_t M = P.M;
  double chunk_mb = 16.0;
  if (g_tune.chunk_mb > 0) chunk_mb = g_tune.chunk_mb;
  int64_t cn = (int64_t)(chunk_mb * 1048576.0 / (32.0 * (double)M));
  if (cn < 1) cn = 1;
  if (cn > n_wf) cn = n_wf;
  P.chunk_n = cn;
  P.pt_threads = M < WS_PT_THREADS ? (int)((M + 31) / 32 * 32) : WS_PT_THREADS;
  P.nblk = (int)((M + P.pt_threads - 1) / P.pt_threads);
  P.onchip = M <= 4096;
  P.G = 1; P.PX = 1; P.lgT = 0;
  if (P.onchip) {
    P.G = (int)(1024 / M); if (P.G < 1) P.G = 1;
  } else {
    if (mode < 2) return WSLDA_EUNSUPPORTED;            // one axis longer than 4096 points
    const int64_t R = M / P.N[0];
    if (R > 8192 || P.N[0] > 1024) return WSLDA_EUNSUPPORTED;
    int64_t px = 4096 / R; if (px < 1) px = 1; if (px > P.N[0]) px = P.N[0];
    P.PX = (int)px;
    int64_t T = 2048 / P.N[0]; if (T < 2) T = 2; if (T > R) T = R;
    P.lgT = ilog2((int)T);
  }
  int64_t dg = (1184 + P.nblk - 1) / P.nblk; if (dg < 1) dg = 1; if (dg > cn) dg = cn;
  P.dG = (int)dg;
  P.nscr = f->current_terms ? 8 : 7;          // + the accumulator of the current / velocity term
  size_t o = 0;
  P.off_tables = o; for (int d = 0; d < 3; ++d) o += align_up((size_t)P.N[d] * 40);       // tw (16) + kk (8) + ko (8) + k^2 natural (8)
  P.off_perwf = o; o += 7 * align_up((size_t)n_wf * 8);
  P.off_fields = o; o += align_up((size_t)DP_COUNT * M * 8) + 12 * align_up((size_t)M * 8) + 2 * align_up((size_t)M * 16);
  P.off_cur = o; if (f->current_terms) o += 3 * align_up((size_t)6 * M * 8);      // A_sigma, v_ext_sigma, W_sigma = A - v: [2][3][M] each
  P.off_obs = o; o += align_up(((size_t)((M + 255) / 256) + 2) * WS_NOBS * 8 + 64);
  P.off_qf = o; if (f->quantum_friction) o += align_up((size_t)2 * M * 8);          // div j_sigma
  P.off_part = o; o += 2 * align_up((size_t)cn * P.nblk * 8);
  P.off_dpart = o; o += align_up((size_t)P.dG * DP_COUNT * M * 8);
  P.scr_bytes = align_up((size_t)cn * 2 * M * 16);
  P.off_scr = o; o += (size_t)P.nscr * P.scr_bytes;
  // fused 3-D path: Ny = Nz = 32, Nx in {8, 16, 32}, Eq. 14 or Eq. 40 operator
  P.fast = mode == 3 && P.N[1] == 32 && P.N[2] == 32 && (P.N[0] == 8 || P.N[0] == 16 || P.N[0] == 32) &&
           f->kin_form != WSLDA_KIN_DIVGRAD &&
           // quantum friction changes the potentials only; its densities (j, B') come from the axis-by-axis kernels on cubic 32^3
           (!f->quantum_friction || (P.N[0] == 32 && !g_tune.disable_persistent && !g_tune.disable_axis_split)) &&
           // the current / velocity coupling is fused only in the matrix-form 32^3 Eq. 40 stage kernels (mega3m.cuh)
           (!f->current_terms || (P.N[0] == 32 && f->kin_form == WSLDA_KIN_SYM40 && g_tune.dmma_stage >= F3M_DEFAULT_ON &&
                                  !g_tune.disable_persistent && !g_tune.disable_axis_split && !g_tune.enable_tma_stage));
  if (g_tune.disable_fused3d) P.fast = 0;
  P.fc = 32; P.ns = 3;
  if (g_tune.fused_chunk > 0) P.fc = g_tune.fused_chunk;
  if (g_tune.fused_streams > 0 && g_tune.fused_streams <= 4) P.ns = g_tune.fused_streams;
  if (P.fc > n_wf) P.fc = (int)n_wf;
  P.off_fast = o; P.fast_spec_bytes = P.fast_part_bytes = P.fast_stream_bytes = 0;
  if (P.fast) {
    P.fast_spec_bytes = align_up((size_t)P.fc * 2 * M * 16);
    P.fast_part_bytes = align_up((size_t)F3_NPART * P.fc * P.N[0] * 8) + align_up((size_t)P.fc * P.nblk * 8) + align_up((size_t)P.fc * 4);
    P.fast_stream_bytes = 3 * P.fast_spec_bytes + P.fast_part_bytes + align_up((size_t)4 * M * 8);
    o += (size_t)P.ns * P.fast_stream_bytes;
  }
  P.mega = P.fast;
  if (g_tune.disable_persistent) P.mega = 0;
  // 32^3: the axis-by-axis stage kernels (mega3s.cuh), whose only ring is Q: large groups
  P.sep = P.mega && P.N[0] == 32;
  if (g_tune.disable_axis_split) P.sep = 0;
  P.gs = P.sep ? 32 : 5;
  if (g_tune.group > 0 && g_tune.group <= 32) P.gs = g_tune.group;
  if (P.gs > n_wf) P.gs = (int)n_wf;
  P.mG = (int)((n_wf + P.gs - 1) / P.gs);
  P.off_mega = o; P.mega_ring_bytes = P.mega_part_bytes = P.mega_acc_bytes = P.mega_sync_bytes = P.mega_pack_bytes = 0;
  if (P.mega) {
    P.mega_ring_bytes = align_up((size_t)F3_RING * P.gs * 2 * M * 16);
    P.mega_part_bytes = align_up((size_t)F3_NPART * n_wf * (P.N[0] < 64 ? 64 : P.N[0]) * 8);   // mega3t: 64 partial sums per spinor
    P.mega_acc_bytes = align_up((size_t)F3_RING * 4 * M * 8);
    P.mega_sync_bytes = align_up(sizeof(F3Sync) + (size_t)5 * n_wf * sizeof(int));      // done[4][G <= n_wf] + one arrival counter per spinor
    P.mega_pack_bytes = align_up((size_t)M * 48) + 32768;            // + the folded derivative matrices of mega3m.cuh (second and first derivative)
    o += 3 * P.mega_ring_bytes + P.mega_part_bytes + P.mega_acc_bytes + P.mega_sync_bytes + P.mega_pack_bytes;
  }
  // (quantum friction changes the potentials only: its densities come from the axis-by-axis kernels beside the stage kernels)
  P.f6 = mode == 3 && P.N[0] == 64 && P.N[1] == 64 && P.N[2] == 64 && f->kin_form == WSLDA_KIN_SYM40 && !f->current_terms &&
         (!f->quantum_friction || !g_tune.disable_axis_split);
  if (g_tune.disable_mega64) P.f6 = 0;
  P.off_f6 = o; P.f6_ring_bytes = P.f6_part_bytes = P.f6_acc_bytes = P.f6_sync_bytes = P.f6_pack_bytes = P.f6_partn_bytes = 0;
  if (P.f6) {
    P.f6_ring_bytes = align_up((size_t)F6_RING * M * 16);
    P.f6_part_bytes = align_up((size_t)F3_NPART * 2 * n_wf * F6_N * 8);
    P.f6_acc_bytes = align_up((size_t)F6_RING * 4 * M * 8);
    P.f6_sync_bytes = align_up(sizeof(F3Sync) + (size_t)5 * 2 * n_wf * sizeof(int));
    P.f6_pack_bytes = align_up((size_t)M * 48);
    P.f6_partn_bytes = align_up((size_t)n_wf * P.nblk * 8);       // norm partials of a whole-batch predictor launch
    o += 3 * P.f6_ring_bytes + P.f6_part_bytes + P.f6_acc_bytes + P.f6_sync_bytes + P.f6_pack_bytes + P.f6_partn_bytes;
  }
  // (the current / velocity coupling is fused only where the matrix-form core exists for it: 64 x 64 and lines of 128)
  P.oc = P.onchip && f->kin_form == WSLDA_KIN_LAPLACE && !f->quantum_friction &&
         (!f->current_terms || (g_tune.dmma_stage >= 0 && ((mode == 2 && P.N[0] == 64 && P.N[1] == 64) || (mode == 1 && P.N[0] == 128))));
  if (g_tune.disable_onchip) P.oc = 0;
  // batch: 64 KB of spinors per CTA (two CTAs per SM) up to 512 points, one spinor per CTA above
  { int64_t S = (M <= 512 ? 4096 : 8192) / (2 * M); if (S < 1) S = 1; if (S > 64) S = 64; if (S > n_wf) S = n_wf; P.ocS = (int)S; }
  { int64_t nb_ = (n_wf + P.ocS - 1) / P.ocS, cap = M <= 512 ? 296 : 148; P.oc_grid = (int)(nb_ < cap ? nb_ : cap); }
  if (g_tune.onchip_ctas > 0 && g_tune.onchip_ctas < P.oc_grid) P.oc_grid = g_tune.onchip_ctas;
  P.off_oc = o; P.oc_dpart_bytes = 0;
  if (P.oc) { P.oc_dpart_bytes = align_up((size_t)P.oc_grid * 4 * (M > 512 ? M : 512) * 8); o += P.oc_dpart_bytes + 131072; }   // + folded derivative matrices (second and first derivative)
  P.total = o;
  return 0;
}

struct wslda_ctx {
  Plan P;
  Lat L;
  double dx[3], dV, Lperp;
  wslda_functional f;
  int m;
  double mu_a, mu_b;
  int lambda_valid;
  wslda_reduce_hook reduce_hook;   // multi-GPU: in-place sum over ranks of the density block (nullable)
  void* reduce_user;
  unsigned raw_local;              // WSLDA_D_* groups of the density block that hold this rank's partial sums (not yet reduced)
  double *kperp2, *cpref, *w_a, *w_b, *scale, *eps, *scale2;
  double* k2n[3];                  // k_d^2 in natural index order
  double hk2[3][64];               // host copy (kernel parameters)
  cudaStream_t aux[4];             // fused path: concurrent chunk streams (created by the library)
  cudaEvent_t ev_fork, ev_join[4];
  cplx *f_spec0[4], *f_spec1[4], *f_X[4];
  cplx *m_spec0, *m_spec1, *m_X;   // persistent-kernel rings
  double *m_part, *m_acc;
  F3Sync* m_sync;
  cplx* m_pack;
  double* oc_dpart;
  double* oc_mat; int oc_dm;       // on-chip 64 x 64: the Laplacian in matrix form on DMMA (onchip_step.cuh), its folded matrices
  cplx *s_spec0, *s_spec1, *s_X, *s_pack;   // 64^3 rings
  double *s_part, *s_acc, *s_partn;
  F3Sync* s_sync;
  int mega_grid;
  int sep_pm, sep_em;              // mega3s.cuh: x-planes per P item, row pairs per XE item
  int sep3;                        // 32^3 Eq. 40: axis-by-axis Laplacian stage kernel (mega3s.cuh)
  int dm3, dm3_grid, dm3_grid_cur; double* m_mat;   // 32^3 Eq. 40: matrix-form (DMMA) stage kernel (mega3m.cuh), its grid, the folded matrices
  int t3, t3_gs, t3_r, t3_ring, t3_lag, t3_grid;    // 32^3 Eq. 40: warp-specialised TMA-fed stage kernel (mega3t.cuh): spinors per group, per heavy super-item
  T3Maps t3_maps;                  // tensor maps of the arrays the library owns (QL ring, alpha); psi is encoded per launch
  int spin_limit;                  // bound of the device-side dependency waits (polls of 200 ns)
  int* err_host;                   // pinned: [0] error word of the last persistent launch, [1] watchdog verdict (copied back asynchronously)
  int* wd_flag;                    // device: watchdog verdict
  double* obs_part; double* obs_out;   // observables: per-block partial sums, result
  double* qf_divj;                 // quantum friction: div j_sigma, [2][M]
  int sticky;                      // a launch could not be made or a device-side wait timed out: every later call fails
  double *f_part[4], *f_partn[4], *f_acc[4];
  int* f_cnt[4];                   // per-spinor arrival counters of k_f3_combine (self-resetting)
  double* raw;
  double *alpha_a, *alpha_b, *V_a, *V_b, *U_a, *U_b, *lap_a, *lap_b, *lambda, *geff, *vext_a, *vext_b;
  cplx *delta, *dext;
  double *cur_A, *cur_v, *cur_W;   // current_terms: [2][3][M] each: A_sigma, v_ext_sigma, W_sigma = A_sigma - v_ext_sigma
  double *part_n, *part_e, *dpart;
  cplx* scr[WS_MAX_SCR];
  int64_t launches;
  // optional per-kernel timing (wslda_profile): event pairs around every launch while enabled
  int prof_on, prof_n;
  std::vector<cudaEvent_t>* prof_ev;
  std::vector<const char*>* prof_name;
  std::vector<double>* prof_work;    // per recorded launch: algorithmic bytes, flops (set with WORK() before LAUNCH)
  double work_bytes, work_flops;
  char err[256];
};

static char g_err[256] = "";
static wslda_status fail(wslda_ctx* c, wslda_status s, const char* msg) {
  snprintf(c ? c->err : g_err, 256, "%s", msg);
  return s;
}
static wslda_status cuda_check(wslda_ctx* c, const char* where) {
  // device-side dependency waits are bounded; a wait that ran out flags the launch, and the flag travels to pinned host
  // memory behind the launch (asynchronously: it is seen by the first call made after that copy has completed)
  if (c && c->err_host && *c->err_host && !c->sticky) {
    c->sticky = 1;
    snprintf(c->err, 256, "a device-side dependency wait timed out in a persistent stage kernel: results since then are invalid");
  }
  if (c && c->err_host && c->err_host[1] && !c->sticky) {
    c->sticky = 2;
    snprintf(c->err, 256, "conservation violated: particle number or total energy left the tolerance given to wslda_watchdog");
  }
  if (c && c->sticky) return c->sticky == 2 ? WSLDA_ESTATE : WSLDA_ECUDA;
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) return WSLDA_OK;
  snprintf(c ? c->err : g_err, 256, "CUDA error at %s: %s", where, cudaGetErrorString(e));
  return WSLDA_ECUDA;
}
#define WS_PROF_MAX 20000
static inline bool prof_begin(wslda_ctx* c, const char* name, cudaStream_t st) {
  if (!c->prof_on || c->prof_n >= WS_PROF_MAX) return false;
  if ((int)c->prof_ev->size() < 2 * (c->prof_n + 1)) {
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    c->prof_ev->push_back(a); c->prof_ev->push_back(b);
  }
  c->prof_name->push_back(name);
  c->prof_work->push_back(c->work_bytes); c->prof_work->push_back(c->work_flops);
  cudaEventRecord((*c->prof_ev)[2 * c->prof_n], st);
  return true;
}
static inline void prof_end(wslda_ctx* c, cudaStream_t st) { cudaEventRecord((*c->prof_ev)[2 * c->prof_n + 1], st); c->prof_n++; }
#define LAUNCHN(c, name, kern, grid, block, smem, st, ...)                             \
  do { bool pr_ = prof_begin(c, name, st); kern<<<grid, block, smem, st>>>(__VA_ARGS__); \
       if (pr_) prof_end(c, st); (c)->launches++; (c)->work_bytes = 0; (c)->work_flops = 0; } while (0)
#define LAUNCH(c, kern, grid, block, smem, st, ...) LAUNCHN(c, #kern, kern, grid, block, smem, st, __VA_ARGS__)
// algorithmic work of the NEXT launch (compulsory HBM bytes: unique full-buffer inputs + outputs; FFT flops as
// 5 N log2 N per line transform) -- only used by the profile report
#define WORK(c, bytes, flops) do { (c)->work_bytes = (double)(bytes); (c)->work_flops = (double)(flops); } while (0)

// stored position p of the in-place DIF transform (radix 8 from L = n down, then the remaining 4 or 2) <-> frequency index
static int ws_fft_radix() { return g_tune.fft_radix == 4 ? 4 : 8; }
static void scrambled_freq(int n, std::vector<int>& fr) {
  fr.resize(n);
  const int maxr = ws_fft_radix();
  for (int p = 0; p < n; ++p) {
    int L = n, rem = p, k = 0, mult = 1;
    while (L > 1) { int r = (L >= maxr) ? maxr : L, sub = L / r, m = rem / sub; rem %= sub; k += m * mult; mult *= r; L = sub; }
    fr[p] = k;
  }
}

extern "C" size_t wslda_workspace_bytes(const int dims[3], wslda_mode mode, int64_t n_wf, const wslda_functional* f) {
  Plan P;
  if (make_plan(dims, (int)mode, n_wf, f, P)) return 0;
  return P.total;
}

extern "C" const char* wslda_last_error(const wslda_ctx* c) { return c ? c->err : g_err; }
extern "C" int64_t wslda_launch_count(const wslda_ctx* c) { return c ? c->launches : 0; }
extern "C" int wslda_history_length(const wslda_ctx* c) { return c ? c->m : 0; }

extern "C" wslda_status wslda_ctx_create(wslda_ctx** out, const int dims[3], const double dx[3], wslda_mode mode,
                                         int64_t n_wf, const wslda_functional* f, void* ws, size_t ws_bytes) {
  if (!out || !dx) return fail(nullptr, WSLDA_EINVAL, "null argument");
  Plan P;
  int rc = make_plan(dims, (int)mode, n_wf, f, P);
  if (rc == WSLDA_EUNSUPPORTED) return fail(nullptr, WSLDA_EUNSUPPORTED, "held lattice sizes must be powers of two >= 2 (and fit the supported regimes)");
  if (rc) return fail(nullptr, WSLDA_EINVAL, "bad dims / mode / n_wf / functional");
  for (int d = 0; d < 3; ++d) if (!(dx[d] > 0)) return fail(nullptr, WSLDA_EINVAL, "dx must be positive");
  if (!ws || ((uintptr_t)ws & 255)) return fail(nullptr, WSLDA_EINVAL, "workspace must be a 256-byte aligned device pointer");
  if (ws_bytes < P.total) return fail(nullptr, WSLDA_ENOMEM, "workspace smaller than wslda_workspace_bytes()");
  wslda_ctx* c = (wslda_ctx*)calloc(1, sizeof(wslda_ctx));
  if (!c) return fail(nullptr, WSLDA_ENOMEM, "host allocation failed");
  c->P = P; c->f = *f;
  c->prof_ev = new std::vector<cudaEvent_t>(); c->prof_name = new std::vector<const char*>();
  c->prof_work = new std::vector<double>();
  c->m = f->ab_order > f->am_order - 1 ? f->ab_order : f->am_order - 1;
  c->spin_limit = 1 << 25;           // ~7 s of polling: far beyond any step, short enough to report a stall
  if (g_tune.spin_limit > 0) c->spin_limit = g_tune.spin_limit;
  cudaMemcpyToSymbol(g_f3_spin_limit, &c->spin_limit, sizeof(int));
  cudaHostAlloc((void**)&c->err_host, 2 * sizeof(int), cudaHostAllocDefault);
  if (c->err_host) c->err_host[0] = c->err_host[1] = 0;
  c->dV = 1.0; c->Lperp = 1.0;
  for (int d = 0; d < 3; ++d) {
    c->dx[d] = dx[d];
    if (d < P.nd) c->dV *= dx[d]; else c->Lperp *= dims[d] * dx[d];
  }
  { const int lgr = ws_fft_radix() == 4 ? 2 : 3; cudaMemcpyToSymbol(g_ws_lgr, &lgr, sizeof(int)); }
  char* base = (char*)ws;
  const int64_t M = P.M;
  Lat& L = c->L;
  L.nd = P.nd; L.M = M; L.invM = 1.0 / (double)M;
  const double PI = 3.14159265358979323846264338327950288;
  size_t o = P.off_tables;
  for (int d = 0; d < 3; ++d) {
    const int n = P.N[d];
    L.N[d] = n; L.lg[d] = P.lg[d];
    std::vector<double> tw(2 * n), kk(n), ko(n), k2(n);
    std::vector<int> fr;
    scrambled_freq(n, fr);
    const double len = n * dx[d];
    for (int j = 0; j < n; ++j) {
      tw[2 * j] = cos(2.0 * PI * j / n); tw[2 * j + 1] = -sin(2.0 * PI * j / n);
      const int l = fr[j];
      double k = (l < n / 2) ? 2.0 * PI * l / len : 2.0 * PI * (l - n) / len;      // Eq. 25
      if (n == 1) k = 0.0;
      kk[j] = k; ko[j] = (n > 1 && l == n / 2) ? 0.0 : k;
      double kn = (j < n / 2) ? 2.0 * PI * j / len : 2.0 * PI * (j - n) / len;       // natural order, Nyquist kept
      if (n == 1) kn = 0.0;
      k2[j] = kn * kn;
      if (j < 64) c->hk2[d][j] = k2[j];
    }
    cplx* dtw = (cplx*)(base + o); double* dkk = (double*)(base + o + (size_t)n * 16); double* dko = dkk + n;
    cudaMemcpy(dtw, tw.data(), (size_t)n * 16, cudaMemcpyHostToDevice);
    cudaMemcpy(dkk, kk.data(), (size_t)n * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(dko, ko.data(), (size_t)n * 8, cudaMemcpyHostToDevice);
    cudaMemcpy(dko + n, k2.data(), (size_t)n * 8, cudaMemcpyHostToDevice);
    c->k2n[d] = dko + n;
    L.tw[d] = dtw; L.kk[d] = dkk; L.ko[d] = dko;
    o += align_up((size_t)n * 40);
  }
  o = P.off_perwf;
  double** pw[7] = {&c->kperp2, &c->cpref, &c->w_a, &c->w_b, &c->scale, &c->eps, &c->scale2};
  for (int q = 0; q < 7; ++q) { *pw[q] = (double*)(base + o); o += align_up((size_t)n_wf * 8); }
  o = P.off_fields;
  c->raw = (double*)(base + o); o += align_up((size_t)DP_COUNT * M * 8);
  double** pf[12] = {&c->alpha_a, &c->alpha_b, &c->V_a, &c->V_b, &c->U_a, &c->U_b, &c->lap_a, &c->lap_b,
                     &c->lambda, &c->geff, &c->vext_a, &c->vext_b};
  for (int q = 0; q < 12; ++q) { *pf[q] = (double*)(base + o); o += align_up((size_t)M * 8); }
  c->delta = (cplx*)(base + o); o += align_up((size_t)M * 16);
  c->dext = (cplx*)(base + o); o += align_up((size_t)M * 16);
  if (f->current_terms) {
    c->cur_A = (double*)(base + P.off_cur); c->cur_v = c->cur_A + 6 * M; c->cur_W = c->cur_v + 6 * M;
    cudaMemset(c->cur_A, 0, (size_t)18 * M * 8);
  }
  c->obs_part = (double*)(base + P.off_obs); c->obs_out = c->obs_part + ((M + 255) / 256) * WS_NOBS;
  c->wd_flag = (int*)(c->obs_out + WS_NOBS);
  if (f->quantum_friction) c->qf_divj = (double*)(base + P.off_qf);
  c->part_n = (double*)(base + P.off_part);
  c->part_e = (double*)(base + P.off_part + align_up((size_t)P.chunk_n * P.nblk * 8));
  c->dpart = (double*)(base + P.off_dpart);
  for (int q = 0; q < P.nscr; ++q) c->scr[q] = (cplx*)(base + P.off_scr + (size_t)q * P.scr_bytes);
  if (P.fast) {
    for (int q = 0; q < P.ns; ++q) {
      char* b = base + P.off_fast + (size_t)q * P.fast_stream_bytes;
      c->f_spec0[q] = (cplx*)b; c->f_spec1[q] = (cplx*)(b + P.fast_spec_bytes); c->f_X[q] = (cplx*)(b + 2 * P.fast_spec_bytes);
      b += 3 * P.fast_spec_bytes;
      c->f_part[q] = (double*)b; c->f_partn[q] = (double*)(b + align_up((size_t)F3_NPART * P.fc * P.N[0] * 8));
      c->f_cnt[q] = (int*)((char*)c->f_partn[q] + align_up((size_t)P.fc * P.nblk * 8));
      cudaMemset(c->f_cnt[q], 0, (size_t)P.fc * 4);
      c->f_acc[q] = (double*)(b + P.fast_part_bytes);
      if (q > 0 || P.ns > 1) cudaStreamCreateWithFlags(&c->aux[q], cudaStreamNonBlocking);
      cudaEventCreateWithFlags(&c->ev_join[q], cudaEventDisableTiming);
    }
    cudaDeviceSynchronize();                               // the counters are zero before any stream of the caller runs
    cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming);
    cudaFuncSetAttribute(k_f3_pass_a<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * F3_TILE_BYTES);
    cudaFuncSetAttribute(k_f3_pass_a<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * F3_TILE_BYTES);
    cudaFuncSetAttribute(k_f3_pass_c<true, F3_APPLY>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * (F3_TILE_BYTES + F3_PLANE * 16));
    cudaFuncSetAttribute(k_f3_pass_c<true, F3_CORR>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * (F3_TILE_BYTES + F3_PLANE * 16));
    cudaFuncSetAttribute(k_f3_pass_c<true, F3_RHS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * (F3_TILE_BYTES + F3_PLANE * 16));
  }
  if (P.mega) {
    char* b = base + P.off_mega;
    c->m_spec0 = (cplx*)b; c->m_spec1 = (cplx*)(b + P.mega_ring_bytes); c->m_X = (cplx*)(b + 2 * P.mega_ring_bytes);
    b += 3 * P.mega_ring_bytes;
    c->m_part = (double*)b; b += P.mega_part_bytes;
    c->m_acc = (double*)b; b += P.mega_acc_bytes;
    c->m_sync = (F3Sync*)b; b += P.mega_sync_bytes;
    c->m_pack = (cplx*)b;
    int occ = 0, best = F3_MEGA_OCC;
#define WS_MEGA_ATTR(K) do { cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * F3_TILE_BYTES); \
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, K, 128, 4 * F3_TILE_BYTES); if (occ > 0 && occ < best) best = occ; } while (0)
    WS_MEGA_ATTR((k_f3_mega<true, F3_APPLY>)); WS_MEGA_ATTR((k_f3_mega<true, F3_CORR>)); WS_MEGA_ATTR((k_f3_mega<true, F3_RHS>));
    WS_MEGA_ATTR((k_f3_mega<false, F3_APPLY>)); WS_MEGA_ATTR((k_f3_mega<false, F3_CORR>)); WS_MEGA_ATTR((k_f3_mega<false, F3_RHS>));
    c->sep3 = P.sep; c->sep_pm = 4; c->sep_em = 2;     // measured: (1,1) 152k, (2,1) 155k, (4,2) 158k spinor-steps/s at 32 per group
    { const int v = g_tune.p_planes; if (v == 1 || v == 2 || v == 4 || v == 8) c->sep_pm = v; }
    { const int v = g_tune.x_rows; if (v == 1 || v == 2 || v == 4) c->sep_em = v; }
    if (c->sep3) {
      WS_MEGA_ATTR((k_f3s_mega<true, F3_APPLY>)); WS_MEGA_ATTR((k_f3s_mega<true, F3_CORR>)); WS_MEGA_ATTR((k_f3s_mega<true, F3_RHS>));
      WS_MEGA_ATTR((k_f3s_mega<false, F3_APPLY>)); WS_MEGA_ATTR((k_f3s_mega<false, F3_CORR>)); WS_MEGA_ATTR((k_f3s_mega<false, F3_RHS>));
    }
#undef WS_MEGA_ATTR
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    c->mega_grid = best * sms;
    // opt-in (measured slower than the mega3s kernels at configs[3]: DESIGN.md 6.5); WSLDA_T3=1 selects it
    c->t3 = 0;
    c->t3 = g_tune.enable_tma_stage && P.sep && f->kin_form == WSLDA_KIN_SYM40;
    c->t3_gs = 8; c->t3_r = 2; c->t3_grid = sms;
    if (g_tune.tma_group > 0 && g_tune.tma_group <= P.gs) c->t3_gs = g_tune.tma_group;
    if (g_tune.tma_block > 1) c->t3_r = g_tune.tma_block;
    if (c->t3_gs > P.gs) c->t3_gs = P.gs;
    while (c->t3_gs % c->t3_r) --c->t3_r;
    if (g_tune.persistent_ctas > 0 && g_tune.persistent_ctas <= sms) c->t3_grid = g_tune.persistent_ctas;
    c->t3_lag = 5; c->t3_ring = 20;                      // ring depth in blocks of r spinors (> 2 lag + the D items' delay)
    if (g_tune.tma_lag > 0) c->t3_lag = g_tune.tma_lag;
    if (g_tune.tma_ring > 1) c->t3_ring = g_tune.tma_ring;
    if ((int64_t)c->t3_ring * c->t3_r > (int64_t)F3_RING * P.gs) c->t3_ring = (int)((int64_t)F3_RING * P.gs / c->t3_r);
    { const int bpg = c->t3_gs / c->t3_r; if (c->t3_ring < 2 * bpg) c->t3_ring = 2 * bpg; }   // a group's blocks + the next group's
    if (c->t3) {
      bool ok = t3_encode_cplx(nullptr, &c->t3_maps.qlX, c->m_spec0, (size_t)c->t3_ring * c->t3_r * 2) &&
                t3_encode_alpha(&c->t3_maps.alP, &c->t3_maps.alX, c->alpha_a, (size_t)((char*)c->alpha_b - (char*)c->alpha_a));
      ok = ok && cudaFuncSetAttribute(k_t3_mega<F3_APPLY>, cudaFuncAttributeMaxDynamicSharedMemorySize, T3_SMEM_BYTES) == cudaSuccess &&
           cudaFuncSetAttribute(k_t3_mega<F3_CORR>, cudaFuncAttributeMaxDynamicSharedMemorySize, T3_SMEM_BYTES) == cudaSuccess &&
           cudaFuncSetAttribute(k_t3_mega<F3_RHS>, cudaFuncAttributeMaxDynamicSharedMemorySize, T3_SMEM_BYTES) == cudaSuccess;
      if (!ok) { cudaGetLastError(); c->t3 = 0; }            // no TMA encoder / not enough shared memory: the mega3s kernels serve
    }
    if (g_tune.persistent_ctas > 0) c->mega_grid = g_tune.persistent_ctas;
    // matrix-form stage kernel (mega3m.cuh): Ce, Co per axis (z, y, x) from the k^2 tables of Eq. 25 (Nyquist kept)
    c->m_mat = (double*)((char*)c->m_pack + align_up((size_t)M * 48));
    c->dm3 = P.sep && f->kin_form == WSLDA_KIN_SYM40 && !c->t3 && g_tune.dmma_stage >= F3M_DEFAULT_ON;
    if (c->dm3) {
      std::vector<double> mat(2 * 3 * 2 * 256);                  // second derivative, then 2 x first derivative (CUR kernels)
      for (int ax = 0; ax < 3; ++ax) {
        const double* k2 = c->hk2[2 - ax];
        double cc[32];
        for (int m = 0; m < 32; ++m) { double t = 0.0; for (int q = 0; q < 32; ++q) t -= k2[q] * cos(2.0 * PI * ((q * m) & 31) / 32.0); cc[m] = t / 32.0; }
        for (int i = 0; i < 16; ++i)
          for (int k = 0; k < 16; ++k) {
            const int m = (i - k) & 31;
            mat[(ax * 2 + 0) * 256 + i * 16 + k] = 0.5 * (cc[m] + cc[(m + 16) & 31]);
            mat[(ax * 2 + 1) * 256 + i * 16 + k] = 0.5 * (cc[m] - cc[(m + 16) & 31]);
          }
      }
      for (int ax = 0; ax < 3; ++ax) {                          // 2 D_d (odd derivative: Nyquist mode dropped), folded once
        const double len = 32 * c->dx[2 - ax];
        double d1[32];
        for (int m = 0; m < 32; ++m) {
          double t = 0.0;
          for (int q = 1; q < 32; ++q) { if (q == 16) continue; const double k = q < 16 ? 2.0 * PI * q / len : 2.0 * PI * (q - 32) / len; t -= k * sin(2.0 * PI * ((q * m) & 31) / 32.0); }
          d1[m] = t / 32.0;
        }
        for (int i = 0; i < 16; ++i)
          for (int k = 0; k < 16; ++k) {
            const int m = (i - k) & 31;
            mat[1536 + (ax * 2 + 0) * 256 + i * 16 + k] = d1[m] + d1[(m + 16) & 31];
            mat[1536 + (ax * 2 + 1) * 256 + i * 16 + k] = d1[m] - d1[(m + 16) & 31];
          }
      }
      {   // fragment order: [axis][Ce | Co][block of 8 rows][k-block][lane = 4 g + t] = M[8 blk + g][4 kb + t] (256 contiguous bytes per warp load)
        std::vector<double> fr(mat.size());
        for (int ae = 0; ae < 12; ++ae)
          for (int blk = 0; blk < 2; ++blk)
            for (int kb = 0; kb < 4; ++kb)
              for (int lane = 0; lane < 32; ++lane)
                fr[ae * 256 + (blk * 4 + kb) * 32 + lane] = mat[ae * 256 + (8 * blk + (lane >> 2)) * 16 + 4 * kb + (lane & 3)];
        mat.swap(fr);
      }
      cudaMemcpy(c->m_mat, mat.data(), mat.size() * 8, cudaMemcpyHostToDevice);
      int occ3 = 0, want = g_tune.dmma_ctas > 0 ? g_tune.dmma_ctas : F3M_OCC, got = want;
      bool ok = true;
#define WS_DM3_ATTR(K) do { ok = ok && cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, F3M_BUF_BYTES) == cudaSuccess; \
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ3, K, 128, F3M_BUF_BYTES); if (occ3 < got) got = occ3; } while (0)
      WS_DM3_ATTR(k_f3m_mega<F3_APPLY>); WS_DM3_ATTR(k_f3m_mega<F3_CORR>); WS_DM3_ATTR(k_f3m_mega<F3_RHS>);
      int got_cur = 2;
      if (f->current_terms) {
        const int keep = got; got = 2;
        WS_DM3_ATTR((k_f3m_mega<F3_APPLY, true>)); WS_DM3_ATTR((k_f3m_mega<F3_CORR, true>)); WS_DM3_ATTR((k_f3m_mega<F3_RHS, true>));
        got_cur = got; got = keep;
        if (got_cur < 1) ok = false;
      }
      c->dm3_grid_cur = got_cur * sms;
#undef WS_DM3_ATTR
      if (!ok || got < 1) { cudaGetLastError(); c->dm3 = 0; }
      if (!c->dm3 && f->current_terms) { snprintf(g_err, 256, "wslda_ctx_create: the fused 32^3 kernels with the current coupling could not be set up"); free(c); return WSLDA_ECUDA; }
      c->dm3_grid = got * sms;
      if (g_tune.persistent_ctas > 0) c->dm3_grid = g_tune.persistent_ctas;
    }
  }
  if (P.f6) {
    char* b = base + P.off_f6;
    c->s_spec0 = (cplx*)b; c->s_spec1 = (cplx*)(b + P.f6_ring_bytes); c->s_X = (cplx*)(b + 2 * P.f6_ring_bytes);
    b += 3 * P.f6_ring_bytes;
    c->s_part = (double*)b; b += P.f6_part_bytes;
    c->s_acc = (double*)b; b += P.f6_acc_bytes;
    c->s_sync = (F3Sync*)b; b += P.f6_sync_bytes;
    c->s_pack = (cplx*)b; b += P.f6_pack_bytes;
    c->s_partn = (double*)b;
    cudaFuncSetAttribute(k_f6_mega<F3_APPLY>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * F6_TILE * 16);
    cudaFuncSetAttribute(k_f6_mega<F3_CORR>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * F6_TILE * 16);
    cudaFuncSetAttribute(k_f6_mega<F3_RHS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * F6_TILE * 16);
  }
  if (P.oc) c->oc_dpart = (double*)(base + P.off_oc);
  c->oc_dm = 0; c->oc_mat = nullptr;
  if (P.oc && P.nd == 2 && P.N[0] == 64 && P.N[1] == 64 && g_tune.dmma_stage >= 0) {
    // second-derivative matrices of Eq. 28b per axis, folded once: [axis][Ce | Co][32][32] (Nyquist mode kept: even derivative)
    c->oc_mat = (double*)(base + P.off_oc + P.oc_dpart_bytes);
    std::vector<double> mat(2 * 2 * 1024);
    for (int ax = 0; ax < 2; ++ax) {
      const double* k2 = c->hk2[ax];
      double cc[64];
      for (int m = 0; m < 64; ++m) { double t = 0.0; for (int q = 0; q < 64; ++q) t -= k2[q] * cos(2.0 * PI * ((q * m) & 63) / 64.0); cc[m] = t / 64.0; }
      for (int i = 0; i < 32; ++i)
        for (int k = 0; k < 32; ++k) {
          const int m = (i - k) & 63;
          mat[(ax * 2 + 0) * 1024 + i * 32 + k] = 0.5 * (cc[m] + cc[(m + 32) & 63]);
          mat[(ax * 2 + 1) * 1024 + i * 32 + k] = 0.5 * (cc[m] - cc[(m + 32) & 63]);
        }
    }
    // first-derivative matrices for the current / velocity coupling (odd derivative: Nyquist mode dropped), same folding
    mat.resize(2 * 2 * 1024 * 2);
    for (int ax = 0; ax < 2; ++ax) {
      const double len = 64 * c->dx[ax];
      double cc[64];
      for (int m = 0; m < 64; ++m) {
        double t = 0.0;
        for (int q = 1; q < 64; ++q) { if (q == 32) continue; const double k = q < 32 ? 2.0 * PI * q / len : 2.0 * PI * (q - 64) / len; t -= k * sin(2.0 * PI * ((q * m) & 63) / 64.0); }
        cc[m] = t / 64.0;
      }
      for (int i = 0; i < 32; ++i)
        for (int k = 0; k < 32; ++k) {
          const int m = (i - k) & 63;
          mat[4096 + (ax * 2 + 0) * 1024 + i * 32 + k] = 0.5 * (cc[m] + cc[(m + 32) & 63]);
          mat[4096 + (ax * 2 + 1) * 1024 + i * 32 + k] = 0.5 * (cc[m] - cc[(m + 32) & 63]);
        }
    }
    {   // fragment order: [axis][Ce | Co][block of 8 rows][k-block][lane = 4 g + t] = M[8 blk + g][4 kb + t]: a warp's load is 256 contiguous bytes
      std::vector<double> fr(mat.size());
      for (int ae = 0; ae < 8; ++ae)
        for (int blk = 0; blk < 4; ++blk)
          for (int kb = 0; kb < 8; ++kb)
            for (int lane = 0; lane < 32; ++lane)
              fr[ae * 1024 + (blk * 8 + kb) * 32 + lane] = mat[ae * 1024 + (8 * blk + (lane >> 2)) * 32 + 4 * kb + (lane & 3)];
      mat.swap(fr);
    }
    cudaMemcpy(c->oc_mat, mat.data(), mat.size() * 8, cudaMemcpyHostToDevice);
    c->oc_dm = 1;
  }
  if (P.oc && P.nd == 1 && P.N[0] == 128 && P.ocS * 2 <= 32 && g_tune.dmma_stage >= 0) {
    // lines of 128 points, folded twice (onchip_step.cuh oc_lap128): Co [64][64], Cee, Ceo [32][32], in fragment order
    c->oc_mat = (double*)(base + P.off_oc + P.oc_dpart_bytes);
    double kk2[128], cc[128], ce[64];
    for (int q = 0; q < 128; ++q) { const double len = 128 * c->dx[0]; const double k = (q < 64) ? 2.0 * PI * q / len : 2.0 * PI * (q - 128) / len; kk2[q] = k * k; }
    for (int m = 0; m < 128; ++m) { double t = 0.0; for (int q = 0; q < 128; ++q) t -= kk2[q] * cos(2.0 * PI * ((q * m) & 127) / 128.0); cc[m] = t / 128.0; }
    for (int m = 0; m < 64; ++m) ce[m] = 0.5 * (cc[m] + cc[m + 64]);        // the even part's circulant (period 64), 1/2 of the first fold
    std::vector<double> mat(4096 + 2 * 1024 + 2 * 4096);
    // fragment order: [block of 8 columns][k-block][lane = 4 g + t] = M[8 blk + g][4 kb + t] (symmetric matrices: column = row)
    for (int blk = 0; blk < 8; ++blk)
      for (int kb = 0; kb < 16; ++kb)
        for (int lane = 0; lane < 32; ++lane) {
          const int i = 8 * blk + (lane >> 2), k = 4 * kb + (lane & 3), m = (i - k) & 127;
          mat[(blk * 16 + kb) * 32 + lane] = 0.5 * (cc[m] - cc[(m + 64) & 127]);
        }
    for (int blk = 0; blk < 4; ++blk)
      for (int kb = 0; kb < 8; ++kb)
        for (int lane = 0; lane < 32; ++lane) {
          const int i = 8 * blk + (lane >> 2), k = 4 * kb + (lane & 3), m = (i - k) & 63;
          mat[4096 + (blk * 8 + kb) * 32 + lane] = 0.5 * (ce[m] + ce[(m + 32) & 63]);
          mat[5120 + (blk * 8 + kb) * 32 + lane] = 0.5 * (ce[m] - ce[(m + 32) & 63]);
        }
    {   // first derivative (odd: Nyquist mode dropped), folded once: De, Do [8 blocks][16 kb][32] at 6144 and 10240
      double d1[128];
      const double len = 128 * c->dx[0];
      for (int m = 0; m < 128; ++m) {
        double t = 0.0;
        for (int q = 1; q < 128; ++q) { if (q == 64) continue; const double k = q < 64 ? 2.0 * PI * q / len : 2.0 * PI * (q - 128) / len; t -= k * sin(2.0 * PI * ((q * m) & 127) / 128.0); }
        d1[m] = t / 128.0;
      }
      for (int blk = 0; blk < 8; ++blk)
        for (int kb = 0; kb < 16; ++kb)
          for (int lane = 0; lane < 32; ++lane) {
            const int i = 8 * blk + (lane >> 2), k = 4 * kb + (lane & 3), m = (i - k) & 127;
            mat[6144 + (blk * 16 + kb) * 32 + lane] = 0.5 * (d1[m] + d1[(m + 64) & 127]);
            mat[10240 + (blk * 16 + kb) * 32 + lane] = 0.5 * (d1[m] - d1[(m + 64) & 127]);
          }
    }
    cudaMemcpy(c->oc_mat, mat.data(), mat.size() * 8, cudaMemcpyHostToDevice);
    c->oc_dm = 2;
  }
  // defaults: zero fields, alpha = 1, w_a = 0, w_b = 1, one mode k_perp = 0 with multiplicity 1, scale = 1
  cudaMemset(base + P.off_perwf, 0, P.off_part - P.off_perwf);
  const int T = 256;
  k_fill<<<(unsigned)((M + T - 1) / T), T>>>(c->alpha_a, M, 1.0);
  k_fill<<<(unsigned)((M + T - 1) / T), T>>>(c->alpha_b, M, 1.0);
  k_fill<<<(unsigned)((n_wf + T - 1) / T), T>>>(c->w_b, n_wf, 1.0);
  k_fill<<<(unsigned)((n_wf + T - 1) / T), T>>>(c->cpref, n_wf, 1.0 / c->Lperp);
  k_fill<<<(unsigned)((n_wf + T - 1) / T), T>>>(c->scale, n_wf, 1.0);
  c->launches += 5;
  cudaFuncSetAttribute(k_gdens_bp<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
  cudaFuncSetAttribute(k_gdens_bp<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
  cudaFuncSetAttribute(k_gdens<32, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
  cudaFuncSetAttribute(k_gdens<32, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
  cudaFuncSetAttribute(k_gdens<32, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
  cudaFuncSetAttribute(k_gdens<64, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
  cudaFuncSetAttribute(k_gdens<64, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
  cudaFuncSetAttribute(k_gdens<64, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * 32 * 128 * 8);
  const int big = 227 * 1024;
  cudaFuncSetAttribute(k_deriv_onchip, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
  cudaFuncSetAttribute(k_planes_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
  cudaFuncSetAttribute(k_planes_inv, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
  cudaFuncSetAttribute(k_xlines, cudaFuncAttributeMaxDynamicSharedMemorySize, big);
  cudaError_t e = cudaDeviceSynchronize();
  if (e != cudaSuccess) {
    snprintf(g_err, 256, "CUDA error in wslda_ctx_create: %s", cudaGetErrorString(e));
    free(c);
    return WSLDA_ECUDA;
  }
  *out = c;
  return WSLDA_OK;
}

// ---- per-kernel timing ------------------------------------------------------------------------------------
extern "C" wslda_status wslda_profile(wslda_ctx* c, int enable) {
  if (!c) return WSLDA_EINVAL;
  if (enable) { c->prof_n = 0; c->prof_name->clear(); c->prof_work->clear(); }
  c->prof_on = enable ? 1 : 0;
  return WSLDA_OK;
}
extern "C" int wslda_profile_report(wslda_ctx* c, char* buf, size_t buf_bytes) {
  if (!c || !buf || !buf_bytes) return -1;
  cudaDeviceSynchronize();
  std::vector<const char*> names; std::vector<double> ms, by, fl, sh; std::vector<long> cnt;
  // launches on concurrent streams overlap in time: besides the raw event-pair duration, attribute every moment of
  // the timeline in equal parts to the launches active in it (the attributed times add up to the busy time)
  const int N = c->prof_n;
  std::vector<double> t0(N), t1(N), share(N, 0.0);
  std::vector<std::pair<double, int>> ends;                      // (time, +(i+1) start | -(i+1) stop)
  for (int i = 0; i < N; ++i) {
    float a = 0.f, b = 0.f;
    cudaEventElapsedTime(&a, (*c->prof_ev)[0], (*c->prof_ev)[2 * i]);
    cudaEventElapsedTime(&b, (*c->prof_ev)[2 * i], (*c->prof_ev)[2 * i + 1]);
    t0[i] = a; t1[i] = (double)a + b;
    ends.push_back({t0[i], i + 1}); ends.push_back({t1[i], -(i + 1)});
  }
  std::sort(ends.begin(), ends.end(), [](const std::pair<double, int>& x, const std::pair<double, int>& y) {
    return x.first < y.first || (x.first == y.first && x.second < y.second); });
  std::vector<int> active;
  for (size_t e = 0; e < ends.size(); ++e) {
    if (e && !active.empty()) {
      const double dt = (ends[e].first - ends[e - 1].first) / (double)active.size();
      for (int i : active) share[i] += dt;
    }
    const int id = ends[e].second;
    if (id > 0) active.push_back(id - 1);
    else for (size_t q = 0; q < active.size(); ++q) if (active[q] == -id - 1) { active[q] = active.back(); active.pop_back(); break; }
  }
  for (int i = 0; i < N; ++i) {
    size_t k = 0;
    while (k < names.size() && strcmp(names[k], (*c->prof_name)[i])) ++k;
    if (k == names.size()) { names.push_back((*c->prof_name)[i]); ms.push_back(0.0); by.push_back(0.0); fl.push_back(0.0); sh.push_back(0.0); cnt.push_back(0); }
    ms[k] += t1[i] - t0[i]; sh[k] += share[i]; cnt[k]++; by[k] += (*c->prof_work)[2 * i]; fl[k] += (*c->prof_work)[2 * i + 1];
  }
  size_t o = 0; buf[0] = 0;
  for (size_t k = 0; k < names.size(); ++k) {
    int w = snprintf(buf + o, buf_bytes - o, "%s %ld %.6f %.6e %.6e %.6f\n", names[k], cnt[k], ms[k], by[k], fl[k], sh[k]);
    if (w < 0 || (size_t)w >= buf_bytes - o) break;
    o += w;
  }
  return (int)names.size();
}

#ifdef F3_TIMING
extern "C" void wslda_debug_cycles(unsigned long long* out, int reset) {
  cudaDeviceSynchronize();
  if (out) cudaMemcpyFromSymbol(out, g_f3_cycles, sizeof(unsigned long long) * 64);
  if (reset) { unsigned long long z[64] = {0}; cudaMemcpyToSymbol(g_f3_cycles, z, sizeof z); }
}
#endif

extern "C" wslda_status wslda_ctx_destroy(wslda_ctx* c) {
  if (!c) return WSLDA_EINVAL;
  if (c->P.fast) {
    for (int q = 0; q < c->P.ns; ++q) { if (c->aux[q]) cudaStreamDestroy(c->aux[q]); cudaEventDestroy(c->ev_join[q]); }
    cudaEventDestroy(c->ev_fork);
  }
  for (cudaEvent_t e : *c->prof_ev) cudaEventDestroy(e);
  delete c->prof_ev; delete c->prof_name; delete c->prof_work;
  if (c->err_host) cudaFreeHost(c->err_host);
  free(c);
  return WSLDA_OK;
}
