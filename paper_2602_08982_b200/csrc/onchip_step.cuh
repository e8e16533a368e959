// onchip_step.cuh -- fused ABM stage kernels for lattices whose spinors fit in shared memory (M <= 4096 points:
// the quasi-1D / quasi-2D modes and small 3-D boxes; configs[0..2]) with the Eq. 14 kinetic operator.
// A CTA keeps a batch of S spinors (S * 2 * M <= 8192 complex128 = 128 KB) on chip for the whole stage:
//   load psi -> forward FFT over the held axes -> -k^2/M (Eq. 26) -> inverse FFT, all in place,
//   pointwise BdG mix (Eqs. 5, 15) -> eps_n = Re <psi|H psi> reduced inside the CTA (Eq. 44b) ->
//   RHS : f = -i (H - eps) psi written once                                        (Alg. 2 step 9)
//   CORR: phi_new = C_part + c0 dt f, its norm reduced inside the CTA, normalised, written once over P,
//         and the densities of phi_new accumulated per CTA in registers             (Alg. 2 steps 3-4, 8)
// so a stage is ONE HBM round trip (read psi [+ C_part], write the result) with no scratch traffic at all.
// Density partials [CTA][4][slots] are summed in a fixed order afterwards: bit-reproducible.
#pragma once
#include "ops.cuh"

enum { OC_APPLY = 0, OC_CORR = 1, OC_RHS = 2 };
#define OC_MAXS 64              // spinors per CTA batch (s_eps / s_sn arrays)
#define OC_SLOTS 8              // (lattice point, spinor) pairs per thread and batch

struct OCArgs {
  Lat L;
  const cplx* psi;             // [n][2][M], first spinor of the call
  const double* scale;         // per spinor, nullable
  const double* kperp2;
  Fields F;
  cplx* out;                   // APPLY: H psi; RHS: f; CORR: phi_new (may alias psi)
  const cplx* cpart;
  double kappa, dV;
  int use_shift, normalize;
  double* eps_out;             // nullable: true eps_n
  int do_dens;
  const double *cpref, *w_a, *w_b;
  double* dpart;               // [gridDim.x][4][slots], slots = max(M, 256)
  int64_t n;
  int S;
};

// per-spinor sums of E[s][i] over the lattice: warp w takes spinors w, w + 8, ...; fixed order
__device__ __forceinline__ void oc_reduce(const double* E, int cnt, int lgM, double* out_s) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, M = 1 << lgM;
  for (int s = warp; s < cnt; s += (blockDim.x >> 5)) {
    double v = 0.0;
    for (int i = lane; i < M; i += 32) v += E[(s << lgM) + i];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) out_s[s] = v;
  }
}

// acc[w mod PT] += (a0..a3) with a register-resident accumulator array: the index is resolved by predication
template <int MAXPT>
__device__ __forceinline__ void oc_dens_acc(double (&acc)[MAXPT][4], int w, int PT, double a0, double a1, double a2, double a3) {
#pragma unroll
  for (int kk = 0; kk < MAXPT; ++kk)
    if ((w & (PT - 1)) == kk) { acc[kk][0] += a0; acc[kk][1] += a1; acc[kk][2] += a2; acc[kk][3] += a3; }
}

// MAXPT = compile-time bound on the lattice points per thread, max(1, M / blockDim.x): 2 (256 threads, M <= 512,
// two CTAs per SM) or 8 (512 threads for M up to 4096, one CTA per SM)
template <int MODE, int MAXPT>
__global__ void __launch_bounds__(MAXPT <= 2 ? 256 : 512, MAXPT <= 2 ? 2 : 1) k_onchip_stage(OCArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Lat& L = a.L;
  const int lgM = L.lg[0] + L.lg[1] + L.lg[2], M = 1 << lgM, S = a.S, tid = threadIdx.x, NT = blockDim.x;
  cplx* F = reinterpret_cast<cplx*>(smem_raw);                       // [S][2][M]
  double* E = reinterpret_cast<double*>(F + (size_t)S * 2 * M);       // [S][M]
  __shared__ double s_eps[OC_MAXS], s_sn[OC_MAXS];
  // slots of this thread: lattice points i(kk) = (tid + 256 kk) & (M - 1), kk < PT; spinors s0, s0 + SSTEP, ...
  const int PT = M >= NT ? M / NT : 1;
  const int SSTEP = M >= NT ? 1 : NT / M, s0 = M >= NT ? 0 : tid >> lgM;
  double acc[MAXPT][4];
#pragma unroll
  for (int kk = 0; kk < MAXPT; ++kk) { acc[kk][0] = acc[kk][1] = acc[kk][2] = acc[kk][3] = 0.0; }
  // work slots of this thread: w -> (kk = w % PT, s = s0 + (w / PT) * SSTEP), at most OC_SLOTS of them; the spinor
  // values of the slots stay in registers from the load to the last phase (psi is read from HBM exactly once)
  const int nsp_full = S > s0 ? (S - s0 + SSTEP - 1) / SSTEP : 0;
  const int64_t n_batches = (a.n + S - 1) / S;
  for (int64_t b = blockIdx.x; b < n_batches; b += gridDim.x) {
    const int64_t n0 = b * S;
    const int cnt = (int)((a.n - n0 < S) ? a.n - n0 : S);
    const int used = cnt * 2 * M;
    const cplx* src = a.psi + (size_t)n0 * 2 * M;
    cplx ru[OC_SLOTS], rv[OC_SLOTS];
#pragma unroll
    for (int w = 0; w < OC_SLOTS; ++w) {
      ru[w] = rv[w] = make_double2(0.0, 0.0);
      if (w < PT * nsp_full) {
        const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
        if (sp < cnt) { ru[w] = __ldg(src + (size_t)(2 * sp) * M + i); rv[w] = __ldg(src + (size_t)(2 * sp + 1) * M + i); }
      }
    }
#pragma unroll
    for (int w = 0; w < OC_SLOTS; ++w) {
      if (w < PT * nsp_full) {
        const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
        if (a.scale && sp < cnt) { const double sc = a.scale[n0 + sp]; ru[w] = cscale(ru[w], sc); rv[w] = cscale(rv[w], sc); }
        F[(2 * sp) * M + i] = ru[w]; F[(2 * sp + 1) * M + i] = rv[w];
      }
    }
    __syncthreads();
    const int G = 2 * S;
    if (L.nd > 2) fft_axis<false>(F, G << (L.lg[0] + L.lg[1]), L.lg[2], 0, L.tw[2]);
    if (L.nd > 1) fft_axis<false>(F, G << L.lg[0], L.lg[1], L.lg[2], L.tw[1]);
    fft_axis<false>(F, G, L.lg[0], L.lg[1] + L.lg[2], L.tw[0]);
    for (int idx = tid; idx < used; idx += NT) {
      const int i = idx & (M - 1);
      const int j2 = i & (L.N[2] - 1), j1 = (i >> L.lg[2]) & (L.N[1] - 1), j0 = i >> (L.lg[1] + L.lg[2]);
      F[idx] = cscale(F[idx], kfactor(L, 0, j0, j1, j2).x);          // -k^2 / M at the stored (digit-reversed) position
    }
    __syncthreads();
    fft_axis<true>(F, G, L.lg[0], L.lg[1] + L.lg[2], L.tw[0]);
    if (L.nd > 1) fft_axis<true>(F, G << L.lg[0], L.lg[1], L.lg[2], L.tw[1]);
    if (L.nd > 2) fft_axis<true>(F, G << (L.lg[0] + L.lg[1]), L.lg[2], 0, L.tw[2]);
    // ---- phase 1: H psi and the integrand of eps_n (F now holds lap u, lap v in natural order).  CORR leaves
    // X = C_part - i kappa H psi in F (phi_new = X + i kappa eps psi once eps_n is known): C_part is consumed here,
    // four slots at a time so that its loads are in flight together without holding 16 more values in registers.
#pragma unroll
    for (int w0 = 0; w0 < OC_SLOTS; w0 += 4) {
      cplx cu[4], cv[4];
      if (MODE == OC_CORR) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          const int w = w0 + r;
          if (w < PT * nsp_full) {
            const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
            if (sp < cnt) { cu[r] = __ldg(a.cpart + (size_t)(2 * (n0 + sp)) * M + i); cv[r] = __ldg(a.cpart + (size_t)(2 * (n0 + sp) + 1) * M + i); }
          }
        }
      }
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const int w = w0 + r;
        if (w < PT * nsp_full) {
          const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
          if (sp < cnt) {
            const int64_t n = n0 + sp;
            const cplx D = cadd(a.F.delta[i], a.F.dext[i]);
            const double pa = a.F.U_a[i] - a.F.mu_a, pb = a.F.U_b[i] - a.F.mu_b, kp2 = a.kperp2[n];
            const cplx u = ru[w], v = rv[w];
            const cplx lu = F[(2 * sp) * M + i], lv = F[(2 * sp + 1) * M + i];
            const cplx Ku = make_double2(-0.5 * lu.x + 0.5 * kp2 * u.x, -0.5 * lu.y + 0.5 * kp2 * u.y);   // Eq. 14
            const cplx Kv = make_double2(-0.5 * lv.x + 0.5 * kp2 * v.x, -0.5 * lv.y + 0.5 * kp2 * v.y);
            const cplx Hu = cadd(Ku, cadd(cscale(u, pa), cmul(D, v)));                                    // Eqs. 5, 15
            const cplx Hv = csub(cmul(cconj(D), u), cadd(Kv, cscale(v, pb)));
            E[(sp << lgM) + i] = u.x * Hu.x + u.y * Hu.y + v.x * Hv.x + v.y * Hv.y;
            if (MODE == OC_APPLY) {
              a.out[(size_t)(2 * n) * M + i] = Hu; a.out[(size_t)(2 * n + 1) * M + i] = Hv;
            } else if (MODE == OC_RHS) {
              F[(2 * sp) * M + i] = Hu; F[(2 * sp + 1) * M + i] = Hv;
            } else {
              F[(2 * sp) * M + i] = make_double2(cu[r].x + a.kappa * Hu.y, cu[r].y - a.kappa * Hu.x);
              F[(2 * sp + 1) * M + i] = make_double2(cv[r].x + a.kappa * Hv.y, cv[r].y - a.kappa * Hv.x);
            }
          }
        }
      }
    }
    __syncthreads();
    oc_reduce(E, cnt, lgM, s_eps);
    __syncthreads();
    if (tid < cnt) {
      const double e_true = a.dV * s_eps[tid];
      if (a.eps_out) a.eps_out[n0 + tid] = e_true;
      s_eps[tid] = (a.use_shift && MODE != OC_APPLY) ? e_true : 0.0;
    }
    __syncthreads();
    if (MODE != OC_APPLY) {
      // ---- phase 2: f = -i (H - eps) psi;  RHS writes it, CORR forms phi_new = C_part + kappa f in place
#pragma unroll
      for (int w = 0; w < OC_SLOTS; ++w) {
        if (w < PT * nsp_full) {
          const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
          if (sp < cnt) {
            const int64_t n = n0 + sp;
            const double e = s_eps[sp];
            const cplx u = ru[w], v = rv[w];
            const cplx Hu = F[(2 * sp) * M + i], Hv = F[(2 * sp + 1) * M + i];
            if (MODE == OC_RHS) {
              const cplx fu = make_double2(Hu.y - e * u.y, -(Hu.x - e * u.x)), fv = make_double2(Hv.y - e * v.y, -(Hv.x - e * v.x));
              a.out[(size_t)(2 * n) * M + i] = fu; a.out[(size_t)(2 * n + 1) * M + i] = fv;
            } else {
              const double ke = a.kappa * e;                           // F holds X: phi_new = X + i kappa eps psi
              const cplx pu = make_double2(Hu.x - ke * u.y, Hu.y + ke * u.x);
              const cplx pv = make_double2(Hv.x - ke * v.y, Hv.y + ke * v.x);
              ru[w] = pu; rv[w] = pv;                                  // phi_new stays in registers
              E[(sp << lgM) + i] = cabs2(pu) + cabs2(pv);
            }
          }
        }
      }
    }
    if (MODE == OC_CORR) {
      __syncthreads();
      oc_reduce(E, cnt, lgM, s_sn);
      __syncthreads();
      if (tid < cnt) s_sn[tid] = a.normalize ? 1.0 / sqrt(a.dV * s_sn[tid]) : 1.0;
      __syncthreads();
      // ---- phase 3: normalise (Alg. 2 step 8), write phi_new once, accumulate its densities (Eqs. 7a, 7b, 7e)
#pragma unroll
      for (int w = 0; w < OC_SLOTS; ++w) {
        if (w < PT * nsp_full) {
          const int i = (tid + NT * (w % PT)) & (M - 1), sp = s0 + (w / PT) * SSTEP;
          if (sp < cnt) {
            const int64_t n = n0 + sp;
            const double sn = s_sn[sp];
            const cplx u = cscale(ru[w], sn), v = cscale(rv[w], sn);
            a.out[(size_t)(2 * n) * M + i] = u; a.out[(size_t)(2 * n + 1) * M + i] = v;
            if (a.do_dens) {
              const double cp = a.cpref[n], wa = a.w_a[n], wb = a.w_b[n], wn = 0.5 * cp * (wb - wa);
              oc_dens_acc<MAXPT>(acc, w, PT, cp * wa * cabs2(u), cp * wb * cabs2(v), wn * (u.x * v.x + u.y * v.y), wn * (u.y * v.x - u.x * v.y));
            }
          }
        }
      }
    }
    __syncthreads();
  }
  if (MODE == OC_CORR && a.do_dens) {
    const int slots = PT * NT;
    double* dp = a.dpart + (size_t)blockIdx.x * 4 * slots;
#pragma unroll
    for (int kk = 0; kk < MAXPT; ++kk)
      if (kk < PT)
#pragma unroll
        for (int f = 0; f < 4; ++f) dp[f * slots + tid + NT * kk] = acc[kk][f];
  }
}

// Alg. 2 steps 1-2 on chip: P = phi + dt sum b_i f_i and C_part = phi + dt sum_{i>=1} c_i f_i in one
// sweep over phi and the history, |P| reduced inside the CTA, the NORMALISED predictor written over phi, C_part over
// the oldest history buffer, and the densities of the predictor accumulated per CTA: 5 reads + 2 writes, nothing else.
struct OCPred {
  Lat L;
  cplx* phi; HistPtrs h; cplx* cpart; AbmCoef k;
  double dV; int normalize;
  int do_dens; const double *cpref, *w_a, *w_b; double* dpart;
  int64_t n; int S;
};

template <int MAXPT>
__global__ void __launch_bounds__(MAXPT <= 2 ? 256 : 512, MAXPT <= 2 ? 2 : 1) k_onchip_pred(OCPred a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Lat& L = a.L;
  const int lgM = L.lg[0] + L.lg[1] + L.lg[2], M = 1 << lgM, S = a.S, tid = threadIdx.x, NT = blockDim.x;
  cplx* F = reinterpret_cast<cplx*>(smem_raw);
  double* E = reinterpret_cast<double*>(F + (size_t)S * 2 * M);
  __shared__ double s_sn[OC_MAXS];
  const int PT = M >= NT ? M / NT : 1;
  const int SSTEP = M >= NT ? 1 : NT / M, s0 = M >= NT ? 0 : tid >> lgM;
  double acc[MAXPT][4];
#pragma unroll
  for (int kk = 0; kk < MAXPT; ++kk) { acc[kk][0] = acc[kk][1] = acc[kk][2] = acc[kk][3] = 0.0; }
  const int64_t n_batches = (a.n + S - 1) / S;
  for (int64_t b = blockIdx.x; b < n_batches; b += gridDim.x) {
    const int64_t n0 = b * S;
    const int cnt = (int)((a.n - n0 < S) ? a.n - n0 : S);
    // work slots of this thread: w -> (kk = w % PT, s = s0 + (w / PT) * SSTEP); two slots per round so that 2 x 2 x (1 + m)
    // independent 16-byte loads are in flight before the first use
    const int nsp = cnt > s0 ? (cnt - s0 + SSTEP - 1) / SSTEP : 0, W = PT * nsp;
    for (int w0 = 0; w0 < W; w0 += 2) {
      cplx ph[2][2], fh[2][2][5];
      size_t off[2][2];
      int si[2], ii[2];
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        const int w = w0 + r < W ? w0 + r : W - 1;               // the tail repeats the last slot (harmless: same values)
        ii[r] = (tid + NT * (w % PT)) & (M - 1); si[r] = s0 + (w / PT) * SSTEP;
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
          off[r][cc] = (size_t)(2 * (n0 + si[r]) + cc) * M + ii[r];
          ph[r][cc] = __ldg(a.phi + off[r][cc]);
#pragma unroll
          for (int j = 0; j < 5; ++j)
            if (j < a.k.ab || j + 1 < a.k.am) fh[r][cc][j] = __ldg(a.h.f[j] + off[r][cc]);
        }
      }
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        if (w0 + r >= W) break;
        double nrm = 0.0;
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
          cplx p = ph[r][cc], q = p;
#pragma unroll
          for (int j = 0; j < 5; ++j) {
            if (j < a.k.ab) { p.x += a.k.b[j] * fh[r][cc][j].x; p.y += a.k.b[j] * fh[r][cc][j].y; }
            if (j + 1 < a.k.am) { q.x += a.k.c[j + 1] * fh[r][cc][j].x; q.y += a.k.c[j + 1] * fh[r][cc][j].y; }
          }
          a.cpart[off[r][cc]] = q;
          F[(2 * si[r] + cc) * M + ii[r]] = p;
          nrm += cabs2(p);
        }
        E[(si[r] << lgM) + ii[r]] = nrm;
      }
    }
    __syncthreads();
    oc_reduce(E, cnt, lgM, s_sn);
    __syncthreads();
    if (tid < cnt) s_sn[tid] = a.normalize ? 1.0 / sqrt(a.dV * s_sn[tid]) : 1.0;
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < MAXPT; ++kk) {
      if (kk < PT) {
        const int i = (tid + NT * kk) & (M - 1);
        for (int s = s0; s < cnt; s += SSTEP) {
          const int64_t n = n0 + s;
          const double sn = s_sn[s];
          const cplx u = cscale(F[(2 * s) * M + i], sn), v = cscale(F[(2 * s + 1) * M + i], sn);
          a.phi[(size_t)(2 * n) * M + i] = u; a.phi[(size_t)(2 * n + 1) * M + i] = v;
          if (a.do_dens) {
            const double cp = a.cpref[n], wa = a.w_a[n], wb = a.w_b[n], wn = 0.5 * cp * (wb - wa);
            acc[kk][0] += cp * wa * cabs2(u);
            acc[kk][1] += cp * wb * cabs2(v);
            acc[kk][2] += wn * (u.x * v.x + u.y * v.y);
            acc[kk][3] += wn * (u.y * v.x - u.x * v.y);
          }
        }
      }
    }
    __syncthreads();
  }
  if (a.do_dens) {
    const int slots = PT * NT;
    double* dp = a.dpart + (size_t)blockIdx.x * 4 * slots;
#pragma unroll
    for (int kk = 0; kk < MAXPT; ++kk)
      if (kk < PT)
#pragma unroll
        for (int f = 0; f < 4; ++f) dp[f * slots + tid + NT * kk] = acc[kk][f];
  }
}

// raw[f][i] = sum over CTAs and duplicate slots of a lattice point, in a fixed order (one warp per output)
__global__ void k_oc_dens_final(const double* dpart, int n_cta, int slots, int64_t M, double* raw) {
  const int64_t o = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (o >= 4 * M) return;
  const int f = (int)(o / M); const int64_t i = o - f * M;
  const int dup = (int)(slots / M), terms = n_cta * dup;
  double s = 0.0;
  for (int t = lane; t < terms; t += 32) {
    const int cta = t / dup, d = t - cta * dup;
    s += dpart[((size_t)cta * 4 + f) * slots + i + (int64_t)d * M];
  }
  for (int k = 16; k > 0; k >>= 1) s += __shfl_xor_sync(0xffffffffu, s, k);
  if (lane == 0) raw[o] = s;
}

// ---- host side ------------------------------------------------------------------------------------------------
static bool g_oc_attr_done = false;
static void oc_launch(wslda_ctx* c, cudaStream_t st, int mode, const cplx* psi, const double* scale, int64_t n0, int64_t n,
                      cplx* out, const cplx* cpart, double kappa, int do_dens, double* eps_user) {
  const Plan& P = c->P;
  OCArgs a;
  a.L = c->L; a.psi = psi; a.scale = scale; a.kperp2 = c->kperp2 + n0; a.F = fields_of(c);
  a.out = out; a.cpart = cpart; a.kappa = kappa; a.dV = c->dV;
  a.use_shift = c->f.subtract_mean_energy; a.normalize = c->f.normalize; a.eps_out = eps_user;
  a.do_dens = do_dens; a.cpref = c->cpref + n0; a.w_a = c->w_a + n0; a.w_b = c->w_b + n0; a.dpart = c->oc_dpart;
  a.n = n; a.S = P.ocS;
  const size_t smem = (size_t)P.ocS * 2 * P.M * 16 + (size_t)P.ocS * P.M * 8;
  if (!g_oc_attr_done) {
    cudaFuncSetAttribute(k_onchip_stage<OC_APPLY, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_CORR, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_RHS, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_APPLY, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_CORR, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_stage<OC_RHS, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    g_oc_attr_done = true;
  }
  const bool small = P.M <= 512;
  const int NT = small ? 256 : 512;
  const int64_t nbat = (n + P.ocS - 1) / P.ocS;
  const int grid = (int)(nbat < P.oc_grid ? nbat : P.oc_grid);
  const double lgM = (double)(P.lg[0] + P.lg[1] + P.lg[2]);
  WORK(c, 32.0 * P.M * n * (mode == OC_CORR ? 3.0 : 2.0), 5.0 * P.M * lgM * 2.0 * 2.0 * n);
  void (*k)(OCArgs);
  if (small) k = mode == OC_APPLY ? k_onchip_stage<OC_APPLY, 2> : mode == OC_CORR ? k_onchip_stage<OC_CORR, 2> : k_onchip_stage<OC_RHS, 2>;
  else k = mode == OC_APPLY ? k_onchip_stage<OC_APPLY, 8> : mode == OC_CORR ? k_onchip_stage<OC_CORR, 8> : k_onchip_stage<OC_RHS, 8>;
  LAUNCHN(c, mode == OC_APPLY ? "k_onchip_apply" : mode == OC_CORR ? "k_onchip_corr" : "k_onchip_rhs", k, grid, NT, smem, st, a);
  if (mode == OC_CORR && do_dens) {
    const int slots = (int)(P.M > NT ? P.M : NT);
    LAUNCH(c, k_oc_dens_final, nb(4 * P.M * 32, 256), 256, 0, st, c->oc_dpart, grid, slots, P.M, c->raw);
  }
}

static wslda_status oc_apply_h(wslda_ctx* c, const cplx* psi, cplx* hpsi, double* eps_dev, int64_t n_first, int64_t n_count,
                               cudaStream_t st) {
  const int64_t M = c->P.M;
  if (n_count > 0)
    oc_launch(c, st, OC_APPLY, psi + 2 * n_first * M, nullptr, n_first, n_count, hpsi + 2 * n_first * M, nullptr, 0.0, 0,
              eps_dev ? eps_dev + n_first : c->eps + n_first);
  return cuda_check(c, "apply_h");
}

static void oc_pred(wslda_ctx* c, cudaStream_t st, cplx* phi, const HistPtrs& h, cplx* cpart, const AbmCoef& k, int do_dens) {
  const Plan& P = c->P;
  OCPred a;
  a.L = c->L; a.phi = phi; a.h = h; a.cpart = cpart; a.k = k; a.dV = c->dV; a.normalize = c->f.normalize;
  a.do_dens = do_dens; a.cpref = c->cpref; a.w_a = c->w_a; a.w_b = c->w_b; a.dpart = c->oc_dpart; a.n = P.n_wf; a.S = P.ocS;
  const size_t smem = (size_t)P.ocS * 2 * P.M * 16 + (size_t)P.ocS * P.M * 8;
  static bool attr = false;
  if (!attr) {
    cudaFuncSetAttribute(k_onchip_pred<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    cudaFuncSetAttribute(k_onchip_pred<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    attr = true;
  }
  const bool small = P.M <= 512;
  const int NT = small ? 256 : 512;
  const int64_t nbat = (P.n_wf + P.ocS - 1) / P.ocS;
  const int grid = (int)(nbat < P.oc_grid ? nbat : P.oc_grid);
  WORK(c, 32.0 * P.M * P.n_wf * (1 + c->m + 2), 0);
  if (small) LAUNCHN(c, "k_onchip_pred", k_onchip_pred<2>, grid, NT, smem, st, a);
  else LAUNCHN(c, "k_onchip_pred", k_onchip_pred<8>, grid, NT, smem, st, a);
  if (do_dens) {
    const int slots = (int)(P.M > NT ? P.M : NT);
    LAUNCH(c, k_oc_dens_final, nb(4 * P.M * 32, 256), 256, 0, st, c->oc_dpart, grid, slots, P.M, c->raw);
  }
}
