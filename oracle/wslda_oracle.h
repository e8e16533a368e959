/*
 * wslda_oracle.h -- CPU oracle for one TDSLDA/BdG time step (TEST INFRASTRUCTURE ONLY).
 *
 * Plain, slow, obviously-correct C99 restatement of the hot path of arXiv 2602.08982 (W-SLDA Toolkit):
 * H*psi with spectral derivatives, densities, pointwise potentials, Adams-Bashforth-Moulton step.
 * complex128 throughout, sequential sums, own radix-2 FFT.  Citations "PAPER.md:<line>" refer to
 * /root/reference/PAPER.md.  This code shares nothing with the CUDA library (no headers, no tables,
 * no helpers); only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load it.  All pointers are HOST pointers owned by the caller unless stated.
 *
 * Pins (tests/test_oracle_*.py): P1-P12, P14-P17 of DESIGN.md section 4.  Unpinned: nothing in this
 * file; the paper's Josephson example is outside the path and is "parity unpinned".
 */
#ifndef WSLDA_ORACLE_H
#define WSLDA_ORACLE_H
#include <stddef.h>
#include <stdint.h>

typedef struct orc_ctx orc_ctx;

typedef struct {
  int    mode;                 /* number of held axes: 3 = full 3D, 2 = quasi-2D (x,y), 1 = quasi-1D (x)   */
  int    dims[3];              /* Nx,Ny,Nz; non-held axes only enter L_perp (Eqs. 29a, 30a)                 */
  double dx[3];
  int64_t n_wf;
  int    func_id;              /* 0 fixed potentials, 1 BdG (Eq. 11), 2 ASLDA (Eq. 12); SLDA = ASLDA p=0    */
  int    force_a1;             /* alpha_sigma = 1 everywhere                              */
  int    spin_symmetric;       /* fold densities per Eq. 8                                */
  int    kin_form;             /* 0 Laplace (Eq. 14), 1 Eq. 40 symmetrised, 2 successive first derivatives   */
  int    ab_order, am_order;   /* (3,4) (4,4) (4,5) (5,5), Eqs. 46-50                                        */
  int    subtract_mean_energy; /* Eq. 44                                                                     */
  int    normalize;            /* Alg. 2 steps 2 and 8                                                       */
  double four_pi_as;           /* BdG coupling C/rho^(1/3) = 4 pi a_s                         */
  double C;                    /* Eq. 12c                                                                    */
  double E_cut;                /* Eq. 22                                                                     */
  int    lambda_mode;          /* 0: Lambda_c recomputed at each potential update; 1: frozen after the first */
  double rho_floor;
  int    current_terms;        /* 1: the current / velocity coupling of Eq. 4c and the j-terms of Eqs. 9b-c */
  int    quantum_friction;     /* 1: the dissipative potentials of Eqs. 66-70 are added at every potential update */
  double qf_alpha, qf_beta, qf_gamma;   /* alpha_qf (Eq. 66), beta_qf, gamma_qf (Eq. 67, 70)                   */
  double qf_rho0, qf_nreq;     /* reference density rho_0 (Eq. 66) and requested particle number N_req (Eq. 70) */
} orc_params;

/* field ids for orc_get_field / orc_set_field */
enum { ORC_RHO_A = 0, ORC_RHO_B = 1, ORC_TAU_A = 2, ORC_TAU_B = 3, ORC_NU = 4 /* complex */,
       ORC_JA_X = 5, ORC_JA_Y = 6, ORC_JA_Z = 7, ORC_JB_X = 8, ORC_JB_Y = 9, ORC_JB_Z = 10,
       ORC_ALPHA_A = 16, ORC_ALPHA_B = 17, ORC_U_A = 18, ORC_U_B = 19, ORC_DELTA = 20 /* complex */,
       ORC_LAP_ALPHA_A = 21, ORC_LAP_ALPHA_B = 22, ORC_LAMBDA_C = 23, ORC_G_EFF = 24, ORC_V_A = 25, ORC_V_B = 26,
       ORC_AA_X = 27, ORC_AA_Y = 28, ORC_AA_Z = 29, ORC_AB_X = 30, ORC_AB_Y = 31, ORC_AB_Z = 32 /* current potentials A_sigma */,
       ORC_BP = 33 /* complex: the kinetic anomalous density B' of Eq. 68 */ };

/* --- transforms (O1) ----------------------------------------------------------------------------------- */
/* in-place radix-2 FFT of n = 2^p complex numbers (interleaved re,im); sign = -1 forward (Eq. 26 convention
 * f~ = sum f exp(-ikx)), +1 inverse (unnormalised).  Returns 0, or -1 if n is not a power of two. */
int  orc_fft1d(double* x, int n, int sign);
/* O(n^2) discrete Fourier transform by its definition, out-of-place; any n. */
void orc_dft1d_naive(const double* in, double* out, int n, int sign);
/* spectral derivatives of one field on the held axes of a lattice (Eqs. 25-26, Nyquist rule PAPER.md:371).
 * in: M complex. lap (nullable): M complex. grad (nullable): mode*M complex, axis-major. */
int  orc_derivatives(int mode, const int dims[3], const double dx[3], const double* in, double* lap, double* grad);

/* --- context --------------------------------------------------------------------------------------------- */
int  orc_create(orc_ctx** ctx, const orc_params* p);
void orc_destroy(orc_ctx* ctx);
/* transverse modes (quasi-1D/2D): kperp[2*m+{0,1}], multiplicity mult[m], spinors [first[m], first[m+1]) */
int  orc_set_modes(orc_ctx*, int n_modes, const double* kperp, const double* mult, const int64_t* first);
int  orc_set_weights(orc_ctx*, const double* w_a, const double* w_b);   /* f_beta(E_n), f_beta(-E_n), frozen */
int  orc_set_mu(orc_ctx*, double mu_a, double mu_b);
int  orc_set_external(orc_ctx*, const double* vext_a, const double* vext_b, const double* delta_ext /* complex, nullable */);
/* external velocity fields v_ext_sigma, [3][M] doubles each (held axes first), nullable = 0 */
int  orc_set_velocity(orc_ctx*, const double* vel_a, const double* vel_b);
int  orc_set_potentials(orc_ctx*, const double* alpha_a, const double* alpha_b, const double* U_a,
                        const double* U_b, const double* delta /* complex */);
int  orc_get_field(orc_ctx*, int field_id, double* dst);
int  orc_set_field(orc_ctx*, int field_id, const double* src);   /* raw densities / Lambda_c, for tests */

/* --- the path ---------------------------------------------------------------------------------------------- */
/* O2/O3: hpsi = H psi for spinors [n_first, n_first+n_count) of the buffer psi (whole-batch base pointers);
 * eps (nullable) receives eps_n = Re dV sum psi^+ H psi.  Eqs. 5, 15, 14, 40, 44b. */
int  orc_apply_h(orc_ctx*, const double* psi, double* hpsi, double* eps, int64_t n_first, int64_t n_count);
/* O4: densities, Eqs. 7/8/29/30; accumulate=0 overwrites, 1 adds to the raw sums. */
int  orc_densities(orc_ctx*, const double* psi, int64_t n_first, int64_t n_count, int accumulate);
/* O5: potentials from the current densities, Eqs. 9-12, 19-22. */
int  orc_update_potentials(orc_ctx*);
/* pointwise functional at one lattice point (exposed for pins P12-P15):
 * in : rho_a, rho_b, tau_a, tau_b, nu(re,im), vext_a, vext_b, lambda_in (used iff use_lambda_in)
 * out: alpha_a, alpha_b, V_a, V_b, delta(re,im), lambda_c, g_eff, energy density (in-scope terms of Eq. 9c) */
int  orc_functional_point(const orc_ctx*, const double in[9], int use_lambda_in, double out[10]);
/* the same with the currents j_a, j_b (3 doubles each): with current_terms the energy density gains
 * sum_sigma (1 - alpha_sigma) j_sigma^2 / (2 rho_sigma) (Eqs. 9b + 9c), V_sigma its derivative, and
 * A_out[0..2] / A_out[3..5] receive the current potentials A_sigma = dE/dj_sigma. */
int  orc_functional_point_j(const orc_ctx*, const double in[9], const double ja[3], const double jb[3], int use_lambda_in,
                            double out[10], double A_out[6]);
/* O7: fill the ABM history: selfstart=0 -> zeros (stationary start), else f(phi_0) and m-1 Taylor steps
 * (Eqs. 52-54).  f_hist: array of m = max(ab_order, am_order-1) buffers, f_hist[0] = newest. */
int  orc_abm_init(orc_ctx*, double* phi, double** f_hist, double dt, int selfstart);
/* O6: one predictor-corrector step following Alg. 2; rotates the roles of f_hist[]. */
int  orc_abm_step(orc_ctx*, double* phi, double** f_hist, double dt);
/* O8 diagnostics: out[0..9] = N_a, N_b, E_kin, E_pot, E_pair, E_pot_ext, E_pair_ext, E_total, E_curr, E_vel_ext
 * (Eqs. 33a-g; E_curr and E_vel_ext, and the -j^2/rho part of E_kin, only with current_terms). */
int  orc_energy(orc_ctx*, double out[10]);
int  orc_history_length(const orc_ctx*);
int  orc_num_threads(void);
#endif
