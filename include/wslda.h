/*
 * wslda.h -- C-ABI boundary of the single-B200 TDSLDA/BdG time-step library (libwslda).
 *
 * One time step of the time-dependent SLDA/BdG equations (arXiv 2602.08982, W-SLDA Toolkit) for a batch of
 * complex128 quasiparticle spinors psi_n = (u_n, v_n) on a periodic lattice:
 *   H psi (spectral kinetic/gradient terms, Eqs. 5, 14, 15, 25-26, 40)  ->  densities (Eqs. 7, 8, 29, 30)
 *   ->  potentials (Eqs. 9-12, 19-22)  ->  Adams-Bashforth-Moulton update (Eqs. 44-50, Alg. 2, Eqs. 52-54).
 * Citations "PAPER.md:<line>" refer to /root/reference/PAPER.md.
 *
 * Conventions (all entry points):
 *  - every array argument named *_dev or documented "device" is a DEVICE pointer owned by the caller
 *    (allocated e.g. with torch); host pointers are documented "host".  The library never frees caller
 *    memory and allocates no device memory of its own: it lives in the workspace given to wslda_ctx_create.
 *  - complex128 is interleaved (re, im).  Spinor buffers are [n][c in {u,v}][ix][iy][iz] contiguous with iz
 *    fastest (loop order PAPER.md:1527-1544), 16-byte aligned; only the held axes (3D: x,y,z; quasi-2D: x,y;
 *    quasi-1D: x) are stored.  Fields are [ix][iy][iz] over the held axes, real (double) or complex.
 *  - every call is asynchronous on the given CUDA stream (a cudaStream_t passed as void*; NULL = default
 *    stream) and returns a status; argument errors return WSLDA_EINVAL before any launch; lattice sizes
 *    that are not powers of two >= 2 return WSLDA_EUNSUPPORTED (the paper needs even sizes);
 *    a CUDA error is reported as WSLDA_ECUDA.  wslda_last_error() gives a text for the last failure.
 *  - the persistent stage kernels wait on device-side completion counters with a bound (wslda_tuning.spin_limit);
 *    a wait that runs out flags its launch, the flag is copied to the host behind the launch, and from the first
 *    call that sees it on every call returns WSLDA_ECUDA ("dependency wait timed out"): results are never
 *    silently wrong, but the report can lag the faulty launch by one call.
 *  - there is no CPU fallback: without a CUDA device every compute call fails with WSLDA_ECUDA.
 */
#ifndef WSLDA_H
#define WSLDA_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wslda_ctx wslda_ctx;   /* opaque; created/destroyed by the library (host object) */

typedef enum { WSLDA_OK = 0, WSLDA_EINVAL = 1, WSLDA_EUNSUPPORTED = 2, WSLDA_ENOMEM = 3, WSLDA_ESTATE = 4,
               WSLDA_ECUDA = 5 } wslda_status;
/* symmetry mode = number of held axes: quasi-1D (Eqs. 30), quasi-2D (Eqs. 29), full 3D */
typedef enum { WSLDA_MODE_1D = 1, WSLDA_MODE_2D = 2, WSLDA_MODE_3D = 3 } wslda_mode;
/* functional: fixed potentials, BdG (Eq. 11), ASLDA (Eq. 12; SLDA = p -> 0) */
typedef enum { WSLDA_FUNC_FIXED = 0, WSLDA_FUNC_BDG = 1, WSLDA_FUNC_ASLDA = 2 } wslda_func_id;
/* kinetic operator: Eq. 14 (alpha = 1), Eq. 40 symmetrised form, successive first derivatives */
typedef enum { WSLDA_KIN_LAPLACE = 0, WSLDA_KIN_SYM40 = 1, WSLDA_KIN_DIVGRAD = 2 } wslda_kin;

typedef struct {
  int func_id;               /* wslda_func_id                                                               */
  int force_a1;              /* alpha_sigma = 1 everywhere, also inside B(p)             */
  int spin_symmetric;        /* fold densities per Eq. 8                                 */
  int kin_form;              /* wslda_kin                                                                   */
  int ab_order, am_order;    /* (3,4) (4,4) (4,5) (5,5): Eqs. 46-50                        */
  int subtract_mean_energy;  /* Eq. 44: evolve with H - <H>_n                                  */
  int normalize;             /* Alg. 2 steps 2 and 8 PAPER.md:646, 652                                      */
  double four_pi_as;         /* BdG coupling C/rho^(1/3) = 4 pi a_s                          */
  double C;                  /* Eq. 12c: -11.11                                                             */
  double E_cut;              /* Eq. 22: default pi^2 / (2 dx^2)                                             */
  int lambda_mode;           /* 0: Lambda_c (Eq. 20) recomputed at every update; 1: frozen after the first  */
  double rho_floor;          /* guard for rho^(1/3) and p at rho -> 0                                       */
  int current_terms;         /* 1: the current / velocity coupling -(i/2){A_sigma - v_ext_sigma, grad} of Eq. 4c
                                 with A_sigma = dE/dj_sigma = (1 - alpha_sigma) j_sigma / rho_sigma
                                 and the j-terms of Eqs. 9b-c in V_sigma.  The
                                anticommutator is applied as W.grad + grad.(W .), both derivatives spectral with the
                                Nyquist rule: exactly Hermitian.  Fused into the matrix-form stage kernels (32^3 with the
                                Eq. 40 operator, 64 x 64, lines of 128 points) whenever the step rebuilds rho and nu
                                only (A_sigma = 0: fixed fields, alpha = 1, BdG); otherwise the general path serves it
                                and wslda_abm_step also rebuilds j at both stages.  0: h of Eq. 4c without it       */
  int quantum_friction;      /* 1: the dissipative potentials of Eqs. 66-70 are added at every
                                potential update: V_sigma += -(qf_alpha / qf_rho0) div j_sigma, Delta += Delta [qf_beta
                                sin(arg nu - arg B') + i qf_gamma (N - qf_nreq) / qf_nreq].  The step then rebuilds j and
                                B' (WSLDA_D_BP) as well: on cubic 32^3 lattices by the axis-by-axis density kernels
                                beside the fused stage kernels, elsewhere on the general path.  Not with FUNC_FIXED  */
  double qf_alpha, qf_beta, qf_gamma;   /* alpha_qf (Eq. 66; 5-10), beta_qf (Eq. 67; about 5), gamma_qf (Eq. 70; about 0.1) */
  double qf_rho0, qf_nreq;   /* reference density rho_0 of Eq. 66, requested particle number N_req of Eq. 70 (> 0)  */
} wslda_functional;

/* field ids for wslda_get_field / wslda_set_field.  Densities are returned folded per Eq. 8 when
 * spin_symmetric is set.  NU and DELTA are complex (M complex128), every other field is M doubles. */
enum { WSLDA_F_RHO_A = 0, WSLDA_F_RHO_B = 1, WSLDA_F_TAU_A = 2, WSLDA_F_TAU_B = 3, WSLDA_F_NU = 4,
       WSLDA_F_JA_X = 5, WSLDA_F_JA_Y = 6, WSLDA_F_JA_Z = 7, WSLDA_F_JB_X = 8, WSLDA_F_JB_Y = 9, WSLDA_F_JB_Z = 10,
       WSLDA_F_ALPHA_A = 16, WSLDA_F_ALPHA_B = 17, WSLDA_F_U_A = 18, WSLDA_F_U_B = 19, WSLDA_F_DELTA = 20,
       WSLDA_F_LAP_ALPHA_A = 21, WSLDA_F_LAP_ALPHA_B = 22, WSLDA_F_LAMBDA_C = 23, WSLDA_F_G_EFF = 24,
       WSLDA_F_V_A = 25, WSLDA_F_V_B = 26,
       WSLDA_F_AA_X = 27, WSLDA_F_AA_Y = 28, WSLDA_F_AA_Z = 29, WSLDA_F_AB_X = 30, WSLDA_F_AB_Y = 31, WSLDA_F_AB_Z = 32
       /* current potentials A_sigma (get only; zero unless current_terms and alpha != 1) */,
       WSLDA_F_BP = 33 /* complex, get only: the kinetic anomalous density B' of Eq. 68 */ };

/* which_mask bits of wslda_densities (Eqs. 7a-g) */
enum { WSLDA_D_RHO = 1u, WSLDA_D_NU = 2u, WSLDA_D_TAU = 4u, WSLDA_D_J = 8u, WSLDA_D_ALL = 15u,
       WSLDA_D_BP = 16u /* B' = -1/2 sum [u lap v^* + v^* lap u] with the weights of nu (Eq. 68); not part of D_ALL */ };

/* Optional tuning of the kernel selection and of the tile / group sizes.  Process-wide: it is read by
 * wslda_workspace_bytes and wslda_ctx_create (contexts that exist keep what they were created with), so set it
 * before sizing the workspace.  A zero field means "library default"; NULL restores all defaults.  None of the
 * fields changes WHAT is computed -- every selectable path is parity-tested against the oracle -- only which
 * kernels compute it (DESIGN.md section 6 says which path serves which lattice and why it is the default). */
typedef struct {
  int disable_fused3d;      /* 1: never use the fused Ny = Nz = 32 kernels (general path everywhere)               */
  int disable_persistent;   /* 1: fused 3-D: chunk pipeline of three passes instead of the persistent stage kernels */
  int disable_axis_split;   /* 1: 32^3: three-pass persistent kernel (mega3d) instead of the axis-by-axis one       */
  int enable_tma_stage;     /* 1: 32^3, Eq. 40: the TMA-fed warp-specialised stage kernel (mega3t; measured slower) */
  int disable_mega64;       /* 1: 64^3: general path instead of the persistent 64^3 kernels                         */
  int disable_onchip;       /* 1: lattices <= 4096 points: general path instead of the fused on-chip stages         */
  int fused_chunk;          /* spinors per chunk of the fused 3-D stage 1 / chunk pipeline (default 32)             */
  int fused_streams;        /* concurrent chunk streams, 1..4 (default 3)                                           */
  int group;                /* spinors per group of the persistent kernels, 1..32 (default 32 at 32^3, else 5)      */
  int p_planes, x_rows;     /* mega3s: x-planes per P item (1, 2, 4, 8; default 4), row pairs per XE item (1, 2, 4; default 2) */
  int persistent_ctas;      /* cap on the persistent grids (default: all SMs x resident CTAs)                       */
  int onchip_ctas;          /* cap on the on-chip stage grids                                                       */
  double chunk_mb;          /* general path: MB of spinors per chunk (default 16)                                   */
  int fft_radix;            /* general on-chip transform: 4 or 8 (default 8)                                        */
  int spin_limit;           /* bound of the device-side dependency waits, in polls of 200 ns (default 2^25, about 7 s);
                               a wait that runs out makes every later call return WSLDA_ECUDA                       */
  int tma_group, tma_block, tma_ring, tma_lag;   /* mega3t: spinors per group (8), per block (2), ring depth in blocks (20),
                               ticks between the P, X, E items of a block (5)                                       */
  int dmma_stage;           /* line derivatives in the matrix form of Eq. 28b on FP64 tensor instructions: the 32^3 Eq. 40
                               stage kernels (mega3m) and the on-chip stage kernels for lines of 128 points and 64 x 64
                               lattices; 0 = library default (on), 1 = on, -1 = off: register / shared-memory FFT kernels */
  int dmma_ctas;            /* mega3m: resident CTAs per SM (default 3)                                             */
} wslda_tuning;
wslda_status wslda_set_tuning(const wslda_tuning* t);

/* Bytes of device workspace wslda_ctx_create needs for this problem (pure host computation; 0 on bad
 * arguments).  dims/dx: host arrays of 3 (Nx,Ny,Nz / dx,dy,dz); non-held axes only enter L_perp (Eqs. 29a, 30a). */
size_t wslda_workspace_bytes(const int dims[3], wslda_mode mode, int64_t n_wf, const wslda_functional* f);

/* Create a context.  dims, dx, f: host.  workspace_dev: device memory of at least wslda_workspace_bytes()
 * bytes, 256-byte aligned, owned by the caller and kept alive until wslda_ctx_destroy.  Builds the k-tables
 * (Eq. 25) and FFT twiddles in the workspace (synchronous copies).  Defaults: weights w_a = 0,
 * w_b = 1; one transverse mode k_perp = 0 with multiplicity 1; mu = 0; alpha = 1; all other fields 0. */
wslda_status wslda_ctx_create(wslda_ctx** ctx, const int dims[3], const double dx[3], wslda_mode mode,
                              int64_t n_wf, const wslda_functional* f, void* workspace_dev, size_t workspace_bytes);
wslda_status wslda_ctx_destroy(wslda_ctx* ctx);

/* Transverse modes (quasi-1D/2D; substitutions PAPER.md:413-419, 444-448).  Host arrays: kperp[2*m+{0,1}],
 * multiplicity mult[m], and mode m owns spinors [first[m], first[m+1]); first[0] = 0, first[n_modes] = n_wf. */
wslda_status wslda_set_modes(wslda_ctx*, int n_modes, const double* kperp, const double* mult, const int64_t* first,
                             void* cuda_stream);
/* Frozen occupation weights f_beta(E_n), f_beta(-E_n); device arrays of n_wf doubles (copied). */
wslda_status wslda_set_weights(wslda_ctx*, const double* w_a_dev, const double* w_b_dev, void* cuda_stream);
/* Chemical potentials: host scalars, read when a later call is enqueued. */
wslda_status wslda_set_mu(wslda_ctx*, double mu_a, double mu_b);
/* External fields (device, nullable = zero): V_ext_sigma real [M], Delta_ext complex [M]. Copied. */
wslda_status wslda_set_external(wslda_ctx*, const double* vext_a_dev, const double* vext_b_dev, const void* delta_ext_dev,
                                void* cuda_stream);
/* External velocity fields v_ext_sigma (a frame moving with v_0, or Omega x r for a rotating frame):
 * device arrays [3][M] doubles each (components along x, y, z; those of non-held axes are ignored), nullable = zero.
 * Copied.  WSLDA_ESTATE unless the context was created with current_terms = 1. */
wslda_status wslda_set_external_velocity(wslda_ctx*, const double* vel_a_dev, const double* vel_b_dev, void* cuda_stream);
/* The setters above copy on the given stream (stream-ordered like every compute call; the host arrays of
 * wslda_set_modes may be freed as soon as it returns). */
/* Fixed potentials (FUNC_FIXED and tests): device arrays alpha_sigma, U_sigma real [M], Delta complex [M];
 * copied; Laplacian of alpha_sigma (Eq. 40) is recomputed spectrally. */
wslda_status wslda_set_potentials(wslda_ctx*, const double* alpha_a_dev, const double* alpha_b_dev,
                                  const double* U_a_dev, const double* U_b_dev, const void* delta_dev, void* cuda_stream);
/* Copy one field to / from caller device memory (see the field id list).  set: raw densities RHO/TAU/NU
 * and LAMBDA_C only (LAMBDA_C also marks the frozen field valid). */
wslda_status wslda_get_field(wslda_ctx*, int field_id, void* dst_dev, void* cuda_stream);
wslda_status wslda_set_field(wslda_ctx*, int field_id, const void* src_dev, void* cuda_stream);

/* hpsi = H psi for spinors [n_first, n_first+n_count) of the whole-batch buffers psi, hpsi (device,
 * [n_wf][2][M] complex128, hpsi != psi); eps_dev (nullable, device, n_wf doubles) receives
 * eps_n = Re dV sum_r psi_n^+ (H psi_n) at index n.  Eqs. 5, 15 PAPER.md:154, 289; Eq. 44b PAPER.md:592. */
wslda_status wslda_apply_h(wslda_ctx*, const void* psi_dev, void* hpsi_dev, double* eps_dev,
                           int64_t n_first, int64_t n_count, void* cuda_stream);
/* Accumulate the densities of spinors [n_first, n_first+n_count) (Eqs. 7a-g, 29b-e, 30b-e) into the
 * context's raw sums; accumulate = 0 overwrites the selected fields, 1 adds (batch streaming). */
wslda_status wslda_densities(wslda_ctx*, const void* psi_dev, int64_t n_first, int64_t n_count,
                             unsigned which_mask, int accumulate, void* cuda_stream);
/* Rebuild alpha_sigma, V_sigma, U_sigma, Lambda_c, g_eff, Delta pointwise from the current densities
 * (Eqs. 9-12, 19-22 PAPER.md:195-255, 311-337) and, for kin_form = SYM40 with a density-dependent alpha,
 * lap(alpha_sigma) spectrally.  FUNC_FIXED: no-op. */
wslda_status wslda_update_potentials(wslda_ctx*, void* cuda_stream);

/* Observables of the state whose densities are in the context (Eqs. 33a-g), computed on the device:
 * obs_dev (device, 10 doubles) = N_a, N_b, E_kin, E_pot, E_pair, E_pot.ext, E_pair.ext, E_total, E_curr, E_vel.ext
 * (the last two, and the -j^2/rho part of E_kin, only with current_terms).  Uses the density block as it stands --
 * call wslda_densities(WSLDA_D_ALL) on the state first (wslda_abm_step refreshes rho and nu only) -- and the current
 * potentials.  Sums are taken in a fixed order: bit-reproducible.  Sharded runs: the block is reduced first. */
enum { WSLDA_OBS_N_A = 0, WSLDA_OBS_N_B, WSLDA_OBS_E_KIN, WSLDA_OBS_E_POT, WSLDA_OBS_E_PAIR, WSLDA_OBS_E_POT_EXT,
       WSLDA_OBS_E_PAIR_EXT, WSLDA_OBS_E_TOTAL, WSLDA_OBS_E_CURR, WSLDA_OBS_E_VEL_EXT, WSLDA_OBS_COUNT };
wslda_status wslda_energy(wslda_ctx*, double* obs_dev, void* cuda_stream);
/* The stability check of the time-dependent codes: computes the observables (into obs_dev,
 * nullable) and compares them ON THE DEVICE with ref_dev (10 doubles from an earlier wslda_energy): if
 * |N_sigma - N_ref| > tol_number N_ref or |E_total - E_ref| > tol_energy |E_ref| (or E is NaN) the context is
 * poisoned -- the verdict travels to the host behind the check, and from the first call that sees it every call
 * returns WSLDA_ESTATE ("conservation violated"), the library's form of "terminate the run".  No host sync. */
wslda_status wslda_watchdog(wslda_ctx*, const double* ref_dev, double tol_number, double tol_energy, double* obs_dev,
                            void* cuda_stream);

/* History length m = max(ab_order, am_order-1). */
int wslda_history_length(const wslda_ctx*);
/* Fill the ABM history for phi (device, [n_wf][2][M], in/out).  f_hist: HOST array of m DEVICE buffers of the
 * same shape, f_hist[0] = newest.  selfstart = 0: zero history (stationary start), potentials
 * rebuilt from phi; else f(phi_0) and m-1 Taylor/midpoint steps (Eqs. 52-54), which advance
 * phi by (m-1) dt.  The roles of f_hist[] are permuted and reported through the same host array. */
wslda_status wslda_abm_init(wslda_ctx*, void* phi_dev, void** f_hist, double dt, int selfstart, void* cuda_stream);
/* One predictor-corrector step following Alg. 2: phi (device) is advanced in place, the
 * oldest history buffer receives f(phi_new) and becomes f_hist[0] (host array permuted in place).  With a
 * self-consistent functional the densities the functional consumes (rho, nu; tau when alpha depends on p)
 * are rebuilt at both stages; j and unused tau are refreshed only by wslda_densities. */
wslda_status wslda_abm_step(wslda_ctx*, void* phi_dev, void** f_hist, double dt, void* cuda_stream);
/* The same step driven from HOST buffers (end-to-end form): copies phi_host and the m host history buffers to
 * the given device buffers, runs wslda_abm_step, copies phi and the new f_hist[0] back and synchronises the
 * stream.  phi_host / f_hist_host[i]: host (pinned for full speed); f_hist_host is permuted like f_hist_dev. */
wslda_status wslda_abm_step_host(wslda_ctx*, void* phi_host, void** f_hist_host, void* phi_dev, void** f_hist_dev,
                                 double dt, void* cuda_stream);
/* Sharding over the spinor index n (the paper's multi-GPU mode): every rank owns
 * a context over its own contiguous range of spinors (with their weights and transverse modes) and the same
 * lattice, functional and external fields.  All step kernels are local; the one exchange is the sum of the
 * density block over the ranks, needed each time a density build is complete and before any potential is formed
 * from it (twice per ABM step, once per Taylor start-up stage, and in wslda_update_potentials / wslda_get_field
 * of a density after wslda_densities).  The hook is called on the HOST, from inside those calls, while their
 * work is being enqueued: it must enqueue, on `cuda_stream`, an IN-PLACE sum over the ranks of `count` doubles at
 * the DEVICE pointer `block` (ncclAllReduce, torch.distributed.all_reduce, ...) and return; it must not
 * synchronise against later work of the same call.  Every rank must make the same sequence of library calls.
 * hook = NULL removes it (single-GPU behaviour).  With a hook installed, wslda_densities(accumulate = 1) onto a
 * block that has already been reduced is WSLDA_EINVAL.  The fixed-potential functional never calls the hook. */
typedef void (*wslda_reduce_hook)(void* user, double* block, int64_t count, void* cuda_stream);
wslda_status wslda_set_reduce_hook(wslda_ctx*, wslda_reduce_hook hook, void* user);
/* Per-kernel device timing for the bench's roofline accounting: while enabled (enable = 1 also clears the
 * record) every kernel launch is bracketed by a CUDA event pair on its own stream (at most 20000 launches are
 * recorded).  wslda_profile_report synchronises the device and writes one line
 *   "kernel_name launches total_ms algorithmic_bytes algorithmic_flops attributed_ms"
 * per kernel into buf (host, buf_bytes long); bytes and flops are the sums of the compulsory HBM bytes and the
 * 5 N log2 N FFT flops the library attributes to those launches; attributed_ms splits every
 * moment of the timeline equally among the launches active in it (launches on concurrent streams overlap, so
 * their raw durations add up to more than the elapsed time).  Returns the number
 * of kernels, -1 on bad arguments. */
wslda_status wslda_profile(wslda_ctx*, int enable);
int wslda_profile_report(wslda_ctx*, char* buf, size_t buf_bytes);
/* Measures the FP64 FMA rate of the current device for the bench's roofline denominator: a kernel of dependent DFMA
 * chains (8 per thread, 2048 threads per SM), best of five timed launches with CUDA events, 2 flops per DFMA.
 * Needs no context; allocates and frees 8 bytes of device memory; synchronises.  flops_per_s: host.  sm_count: host,
 * nullable. */
wslda_status wslda_fp64_probe(double* flops_per_s, double* sm_count);
/* Allocation-free gradient densities, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops): tau_sigma = sum_n cw^sigma_n |grad w_n|^2 (Eqs. 7c-d) and
 * j_a = -sum_n cw^a_n Im[u_n grad u_n^*], j_b = +sum_n cw^b_n Im[v_n grad v_n^*] (Eqs. 7f-g) of n_wf
 * spinors on a cubic periodic lattice of side 32 or 64 (full 3-D; spectral first derivative of Eq. 26 with the Nyquist mode
 * dropped).  Needs no context and no workspace: the partial planes of the axis-by-axis kernel live in a
 * file-scope device array of wslda_static_scratch_bytes() = 24 MiB that every GPU loading the library holds until exit.
 * No cudaMalloc / cudaFree / allocating library call is made, on the first call or later (the first call on a device looks
 * up the array's device address and sets a kernel attribute).  ALL calls on a device share that array: two calls that may
 * overlap on the GPU (different streams without an ordering between them, concurrent host threads) race; calls on one
 * stream are safe.  The array keeps the last call's contents; nothing in it has to start at zero.
 *   psi   device, complex128 [n_wf][2][n_side][n_side][n_side] (z fastest), read only
 *   cw_a, cw_b  device, double [n_wf]: c_n w^a_n and c_n w^b_n -- the prefactor of Eqs. 29-30 (1 in full 3-D) times the
 *         weight of Eq. 7 / Eq. 8
 *   dx    host, 3 lattice spacings
 *   tau   device, double [2][M] (a, b), M = n_side^3; nullable.   j: device, double [2][3][M] (a: x, y, z; b: x, y, z); nullable
 * Asynchronous on `stream`; outputs are overwritten (no accumulate).  Sums run over n in increasing order inside
 * min(n_wf, 8 | 1) groups (32^3 | 64^3) added in index order: bit-reproducible.  Errors (message through
 * wslda_last_error(NULL)): WSLDA_EINVAL for null pointers, n_side beyond WSLDA_STATIC_MAX_SIDE or not 32 / 64, n_wf outside
 * [1, WSLDA_STATIC_MAX_SPINORS], non-positive dx; WSLDA_ECUDA when there is no device or a launch fails. */
#define WSLDA_STATIC_MAX_SIDE 64
#define WSLDA_STATIC_MAX_SPINORS 65536
size_t wslda_static_scratch_bytes(void);
wslda_status wslda_gradient_densities_static(const void* psi, const double* cw_a, const double* cw_b, int64_t n_wf, int n_side,
                                             const double dx[3], double* tau, double* j, void* cuda_stream);
/* Number of kernels this context has launched so far (for the bench's gpu_launches claim). */
int64_t wslda_launch_count(const wslda_ctx*);
const char* wslda_last_error(const wslda_ctx*);

#ifdef __cplusplus
}
#endif
#endif
