// mega3t.cuh -- 32^3 stage kernels, Eq. 40 operator: warp-specialised persistent dataflow fed by TMA.
//
// Same mathematics as mega3s.cuh (the spectral Laplacian of Eq. 26, taken axis by axis; Eq. 40,
// PAPER.md:561-565; the BdG mix of Eqs. 5/15; Alg. 2 steps 3-4, 8, 9), but the
// work of a stage is split by what it needs from the SM:
//   HEAVY warps (8 per SM, 192 registers, in 4 pairs) hold one 32-point complex128 line per thread and do nothing but
//     shared memory -> registers -> FFT, -k^2, inverse FFT -> shared memory / one coalesced store.  Their inputs are
//     brought into shared-memory tiles by TMA tensor copies (cp.async.bulk.tensor, SASS UTMALDG) completing on
//     mbarriers, issued by a LOADER lane for the NEXT item as soon as the current item has lifted its lines out of
//     the tile, so no heavy warp ever waits on a global load or on a ticket.
//       P (n, c, x-plane): Q_c = alpha_c (d_y^2 + d_z^2) w + (d_y^2 + d_z^2)(alpha_c w)        -> QL ring
//       X (n, c, y-row)  : L_c = Q_c + alpha_c d_x^2 w + d_x^2 (alpha_c w)   (in place)        -> QL ring
//     warp t = 0 of a pair transforms w, warp t = 1 transforms alpha_c w, both from ONE staged copy of psi and one
//     staged copy of alpha_c (kept across the `r` spinors of a super-item).  Plane tiles are stored with the 128-byte
//     TMA swizzle, so the z-lines (thread = y) and the y-lines (thread = z) are both read without bank conflicts from
//     unpadded 16 KB tiles: 4 pairs x (3 x 16 KB + 8 KB) = 224 KB of the SM's 227 KB.
//   LIGHT warps (64 registers) stream: the pointwise epilogue E (K = -L/4 + ..., BdG mix, eps_n / norm partial
//     sums, stage combination -> X ring or H psi) and the per-group closing items D (final combination with eps_n and
//     the norm, densities) -- plain coalesced loads, many warps to hide their latency, no line registers to park.
// Register budgets are moved between the kinds with setmaxnreg (512 threads x 128 at launch -> 192 / 64).
// Dispatch: two atomic ticket streams (heavy: P, X; light: E, D) in pipeline order; an item waits only for items with
// smaller tickets, which running warps hold, so the scheme cannot deadlock; counters use red.release / ld.acquire.
#pragma once
#include <cuda.h>
#include "mega3s.cuh"
#include "async_copy.cuh"

#define T3_PAIRS 4
#define T3_LIGHT 8                                  // light warps per CTA (warp 8 lends lanes 0..3 as loaders)
#define T3_THREADS (64 * T3_PAIRS + 32 * T3_LIGHT)  // 512
#define T3_TILE_BYTES 16384                         // one 32 x 32 complex128 tile
#define T3_AL_BYTES 8192                            // one 32 x 32 double tile
#define T3_PAIR_BYTES (3 * T3_TILE_BYTES + T3_AL_BYTES)
#define T3_MISC_OFF (T3_PAIRS * T3_PAIR_BYTES)      // 229376: mbarriers, mailboxes
#define T3_MISC_BYTES 2048
#define T3_SMEM_BYTES (T3_MISC_OFF + T3_MISC_BYTES)
#define T3_EPL 1                                    // x-planes per E ticket (one completion signal per ticket)
#define T3_HEAVY_REGS 192
#define T3_LIGHT_REGS 64

// optional phase timing (-DT3_TIMING): per-warp cycle sums in shared memory (no contention), flushed by the kernel
#ifdef T3_TIMING
#define T3_T0() long long t_ = clock64()
#define T3_T(kind, phase) do { long long n_ = clock64(); if (p.lane == 0) p.cyc[(kind) * 8 + (phase)] += (unsigned long long)(n_ - t_); t_ = n_; } while (0)
#else
#define T3_T0() do {} while (0)
#define T3_T(kind, phase) do {} while (0)
#endif

#ifdef T3_TIMING
__device__ unsigned long long g_t3_cycles[2][16];
__device__ unsigned long long g_t3_prof[16];
#define T3_P0() long long tp_ = clock64()
#define T3_P(slot) do { long long n_ = clock64(); pr_[slot] += (unsigned long long)(n_ - tp_); tp_ = n_; } while (0)
#else
#define T3_P0() do {} while (0)
#define T3_P(slot) do {} while (0)
#endif

// ---- TMA tensor copies ----------------------------------------------------------------------------------------
__device__ __forceinline__ void t3_tma3(uint32_t dst, const CUtensorMap* m, int c0, int c1, int c2, uint32_t bar, uint64_t pol) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;"
               :: "r"(dst), "l"(m), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ void t3_tma4(uint32_t dst, const CUtensorMap* m, int c0, int c1, int c2, int c3, uint32_t bar, uint64_t pol) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4, %5}], [%6], %7;"
               :: "r"(dst), "l"(m), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar), "l"(pol) : "memory");
}

// The five views of the stage's arrays (encoded on the host per launch, ctx side: t3_encode_maps):
//   psiP : psi as planes   (64 dbl [z, contiguous], 32 y, planes = 2 n_wf * 32)      box {16, 32, 1}   swizzle 128B
//   alP  : alpha as planes (32 dbl [z], 32 y, 32 x, 2 components)                    box {16, 32, 1, 1} swizzle 128B
//   psiX : psi as rows     (64 dbl [z], 32 y, 32 x, 2 n_wf components)               box {64, 1, 32, 1} no swizzle
//   qlX  : the QL ring, same view as psiX
//   alX  : alpha as rows   (32 dbl [z], 32 y, 32 x, 2 components)                    box {32, 1, 32, 1} no swizzle
struct T3Maps { CUtensorMap psiP, alP, psiX, qlX, alX; };

typedef CUresult (*T3EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                               const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
// the driver's encoder, looked up once through the runtime (no link against libcuda)
static T3EncodeFn t3_encoder() {
  static T3EncodeFn fn = nullptr;
  if (!fn) {
    cudaDriverEntryPointQueryResult q;
    void* p = nullptr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) fn = (T3EncodeFn)p;
  }
  return fn;
}
static bool t3_encode(CUtensorMap* m, const void* base, int rank, const cuuint64_t* dims, const cuuint64_t* strides, const cuuint32_t* box, bool swz) {
  T3EncodeFn f = t3_encoder();
  if (!f) return false;
  const cuuint32_t es[5] = {1, 1, 1, 1, 1};
  return f(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, (cuuint32_t)rank, const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
           swz ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}
// views of a spinor array of `ncomp` components ([ncomp][32][32][32] complex128): planes (swizzled) and rows
static bool t3_encode_cplx(CUtensorMap* planes, CUtensorMap* rows, const void* base, size_t ncomp) {
  bool ok = true;
  if (planes) { const cuuint64_t d[3] = {64, 32, ncomp * 32}, st[2] = {512, 16384}; const cuuint32_t b[3] = {16, 32, 1}; ok = ok && t3_encode(planes, base, 3, d, st, b, true); }
  if (rows) { const cuuint64_t d[4] = {64, 32, 32, ncomp}, st[3] = {512, 16384, 524288}; const cuuint32_t b[4] = {64, 1, 32, 1}; ok = ok && t3_encode(rows, base, 4, d, st, b, false); }
  return ok;
}
// views of the two real alpha fields (alpha_b = alpha_a + comp_stride bytes)
static bool t3_encode_alpha(CUtensorMap* planes, CUtensorMap* rows, const void* alpha_a, size_t comp_stride) {
  const cuuint64_t d4[4] = {32, 32, 32, 2}, s4[3] = {256, 8192, comp_stride};
  const cuuint32_t bp[4] = {16, 32, 1, 1}, br[4] = {32, 1, 32, 1};
  return t3_encode(planes, alpha_a, 4, d4, s4, bp, true) && t3_encode(rows, alpha_a, 4, d4, s4, br, false);
}

// byte offset of complex element (row r, column c) of a plane tile under the 128-byte swizzle of its four 4 KB
// column blocks (c >> 3): 16-byte chunk (c & 7) of the 128-byte row r is stored at chunk (c & 7) ^ (r & 7)
__device__ __forceinline__ int t3_swz16(int r, int c) { return ((c >> 3) << 12) + (r << 7) + ((((c & 7) ^ r) & 7) << 4); }
// same for a double tile (two 4 KB column blocks c >> 4; chunk (c >> 1) & 7; half (c & 1))
__device__ __forceinline__ int t3_swz8(int r, int c) { return ((c >> 4) << 12) + (r << 7) + (((((c >> 1) & 7) ^ r) & 7) << 4) + ((c & 1) << 3); }

struct T3Bars {                 // per pair, in shared memory
  uint64_t fullA, fullQ, fullAL;        // TMA landed: A tile, Q tile (X items, into B1), alpha tile
  uint64_t emptyA;                      // both warps have lifted their last lines out of A        (count 2)
  uint64_t itemdone;                    // both warps are through with every tile of the item      (count 2)
  uint64_t hready, hfree;               // hand-off tile (P: B1, t=1 -> t=0; X: B0, t=0 -> t=1) written / consumed
  uint64_t mail;                        // a mailbox slot was filled (count 1, loader)
};
struct T3Mail {                 // what the loader tells the pair about an item
  int kind;                     // 0 P, 1 X, -1 exit
  int n;                        // spinor (index into the launch's arrays)
  int c, idx;                   // component, x-plane (P) or y-row (X)
  int slot;                     // ring component index ((g % R) * gs + nl) * 2 + c
  int new_alpha;                // the alpha tile was restaged for this item
  int done_idx;                 // completion counter to bump after the item's stores, or -1
  int pad;
  double s;                     // the spinor's scale (psi is used as s * psi)
};

struct T3Pair {
  unsigned char* base;          // the pair's shared memory: A | B0 | B1 | AL
  T3Bars* bars;
  uint32_t phA, phQ, phAL, phH, phF, phM;      // parities
  int t, lane;
#ifdef T3_TIMING
  unsigned long long* cyc;      // [2][8] per-warp phase counters in shared memory
#endif
};
#define T3_A(p) ((p).base)
#define T3_B0(p) ((p).base + T3_TILE_BYTES)
#define T3_B1(p) ((p).base + 2 * T3_TILE_BYTES)
#define T3_AL(p) ((p).base + 3 * T3_TILE_BYTES)
#define T3_C(ptr, off) (*reinterpret_cast<cplx*>((ptr) + (off)))
#define T3_D(ptr, off) (*reinterpret_cast<double*>((ptr) + (off)))

// ---- the two heavy item kinds, written around ONE instance of the line transform (instruction-cache footprint: the
// warps of an SM are in different phases of different items, so the hot code has to stay small) ----------------------
// P (kind 0): the pair leaves Q_c of one x-plane in the ring: step 0 = z-lines (thread = y), step 1 = y-lines (thread = z).
// X (kind 1): L_c = Q_c + alpha d_x^2 w + d_x^2 (alpha w) for one y-row, in place in the ring; A = psi rows [x][z], AL =
//             alpha rows [x][z], B1 = the Q rows (all row-major, lane = z: conflict-free as they are).
__device__ __forceinline__ void t3_body_px(T3Pair& p, int kind, cplx* out, double s, const double* k2all, const F3Pol& pol, cplx* x) {
  const int lane = p.lane, t = p.t;
  unsigned char* A = T3_A(p); unsigned char* AL = T3_AL(p); unsigned char* B0 = T3_B0(p); unsigned char* B1 = T3_B1(p);
  unsigned char* B = t ? B1 : B0;
  T3_T0();
#pragma unroll 1
  for (int step = kind; step < 2; ++step) {                     // P: steps 0, 1; X: step 1 only
    if (kind == 0 && step == 0) {                               // z-lines: thread = y, register index = z
#pragma unroll
      for (int j = 0; j < F3_N; ++j) x[j] = T3_C(A, t3_swz16(lane, j));
      if (t) {
#pragma unroll
        for (int j = 0; j < F3_N; j += 2) {
          const double2 a2 = *reinterpret_cast<const double2*>(AL + t3_swz8(lane, j));
          x[j] = cscale(x[j], a2.x); x[j + 1] = cscale(x[j + 1], a2.y);
        }
      }
    } else {
      if (kind == 0) {                                          // y-lines: thread = z, register index = y
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = T3_C(A, t3_swz16(j, lane));
        if (t) {
#pragma unroll
          for (int j = 0; j < F3_N; ++j) x[j] = cscale(x[j], T3_D(AL, t3_swz8(j, lane)));
        }
      } else {                                                  // x-lines: thread = z, register index = x
#pragma unroll
        for (int j = 0; j < F3_N; ++j) x[j] = T3_C(A, (j * F3_N + lane) * 16);
        if (t) {
#pragma unroll
          for (int j = 0; j < F3_N; ++j) x[j] = cscale(x[j], T3_D(AL, (j * F3_N + lane) * 8));
        }
      }
      __syncwarp();
      if (lane == 0) ac_mbar_arrive(ac_smem(&p.bars->emptyA));    // A is consumed by this warp
    }
    T3_T(kind, 2);
    const int kb = kind ? 64 : step * 32;
    f3s_d2(x, [&](int j) { return k2all[kb + j]; }, s);
    T3_T(kind, 4);
    if (kind == 0 && step == 0) {
      if (t) { ac_mbar_wait(ac_smem(&p.bars->hfree), p.phF ^ 1); }   // B1 of the previous item has been read by the partner
#pragma unroll
      for (int j = 0; j < F3_N; ++j) T3_C(B, t3_swz16(lane, j)) = x[j];
      __syncwarp();
      T3_T(0, 5);
    }
  }
  if (kind == 0) {
#pragma unroll
    for (int j = 0; j < F3_N; ++j) { const cplx z = T3_C(B, t3_swz16(j, lane)); x[j] = cadd(x[j], z); }
    T3_T(0, 5);
    if (t) {                                                    // (d_y^2 + d_z^2)(alpha w): hand it to the partner in B1
      __syncwarp();
#pragma unroll
      for (int j = 0; j < F3_N; ++j) T3_C(B, (j * F3_N + lane) * 16) = x[j];
      __syncwarp();
      if (lane == 0) ac_mbar_arrive(ac_smem(&p.bars->hready));
    } else {
#pragma unroll
      for (int j = 0; j < F3_N; ++j) x[j] = cscale(x[j], T3_D(AL, t3_swz8(j, lane)));
      ac_mbar_wait(ac_smem(&p.bars->hready), p.phH);
#pragma unroll
      for (int j = 0; j < F3_N; ++j) st_pol(out + j * F3_N + lane, cadd(x[j], T3_C(B1, (j * F3_N + lane) * 16)), pol.keep);
      __syncwarp();
      if (lane == 0) ac_mbar_arrive(ac_smem(&p.bars->hfree));
    }
  } else {
    if (t == 0) {                                               // alpha d_x^2 w + Q  -> B0
      ac_mbar_wait(ac_smem(&p.bars->fullQ), p.phQ);
      ac_mbar_wait(ac_smem(&p.bars->hfree), p.phF ^ 1);         // B0 of the previous item has been read by the partner
      T3_T(1, 7);
#pragma unroll
      for (int j = 0; j < F3_N; ++j) {
        const double a = T3_D(AL, (j * F3_N + lane) * 8);
        const cplx qv = T3_C(B1, (j * F3_N + lane) * 16);
        T3_C(B0, (j * F3_N + lane) * 16) = make_double2(fma(a, x[j].x, qv.x), fma(a, x[j].y, qv.y));
      }
      __syncwarp();
      if (lane == 0) ac_mbar_arrive(ac_smem(&p.bars->hready));
    } else {
      ac_mbar_wait(ac_smem(&p.bars->hready), p.phH);
      T3_T(1, 7);
#pragma unroll
      for (int j = 0; j < F3_N; ++j) st_pol(out + (size_t)j * F3_PLANE + lane, cadd(x[j], T3_C(B0, (j * F3_N + lane) * 16)), pol.keep);
      __syncwarp();
      if (lane == 0) ac_mbar_arrive(ac_smem(&p.bars->hfree));
    }
    p.phQ ^= 1;
  }
  p.phH ^= 1; p.phF ^= 1;
  T3_T(kind, 6);
}

// ---- the stage kernel --------------------------------------------------------------------------------------------
struct T3Sync {                 // device counters, zeroed before every launch; followed by doneP[NB] doneX[NB] doneE[NB] doneS[G] doneD[G]
  int nextH, nextL;             // heavy / light tickets
  int error;                    // a bounded dependency wait ran out (sticky for the launch; copied to the host afterwards)
  int pad;
};
struct T3Mega {
  F3Mega m;                     // arrays, scalars and flags as in mega3d.cuh; spec0 = QL ring, X = X ring, m.sync unused;
                                // m.part = [F3_NPART][n * 64] partial sums per (spinor, x-plane, warp of the pair)
  T3Sync* sync;
  double* sn_out;               // per spinor: 1 / |phi_new| (CORR)
  double* eps_user;             // APPLY: second copy of eps_n for the caller (nullable)
  double k2all[96];             // k_z^2, k_y^2, k_x^2, natural order
  int gs, r, G, R, RA, lag;     // spinors per group (a multiple of r), per block; groups; ring depth in blocks (QL, X); density ring slots;
                                // ticks between the P, X and E items of a block in the heavy ticket stream
  int spin_limit;               // bound of the dependency waits, in polls of 200 ns
};

__device__ __forceinline__ void t3_wait(const int* ctr, int target, T3Sync* sy, int limit) {
  int spins = 0;
  while (f3_ld_acquire(ctr) < target) {
    __nanosleep(200);
    if (++spins > limit) { sy->error = 1; break; }
  }
}

// Dependencies are tracked per BLOCK of r spinors (the heavy super-item unit), so that a block flows P -> X -> E as soon
// as its own items are through, and only the closing D items (register accumulation of the densities over a group) wait
// for a whole group: the latency of a block, not of a group, sets how many spinors have to be in flight (ring slots).
// Counters after T3Sync: doneP[NB] doneX[NB] doneE[NB] doneS[G] doneD[G], NB = ceil(n / r) blocks, G groups of gs.
// Heavy ticket stream, tick t: P(t) [64 super-items (c, plane)], X(t - lag) [64], E(t - 2 lag) [r * 32 / T3_EPL].
__device__ __forceinline__ int t3_nb(const T3Mega& A) { return (A.m.n + A.r - 1) / A.r; }

// loader lane of pair `pr`: draws the tickets, waits for their dependencies, stages the tiles, fills the mailbox
template <int MODE>
__device__ __forceinline__ void t3_loader(const T3Maps& maps, const T3Mega& A, unsigned char* smem, int pr) {
  const F3Mega& a = A.m;
  const F3Pol pol = f3_policies();
  T3Bars* b = reinterpret_cast<T3Bars*>(smem + T3_MISC_OFF) + pr;
  T3Mail* mail = reinterpret_cast<T3Mail*>(smem + T3_MISC_OFF + T3_PAIRS * sizeof(T3Bars)) + pr * 2;
  unsigned char* base = smem + pr * T3_PAIR_BYTES;
  const uint32_t sA = ac_smem(base), sB1 = ac_smem(base + 2 * T3_TILE_BYTES), sAL = ac_smem(base + 3 * T3_TILE_BYTES);
  const uint32_t bA = ac_smem(&b->fullA), bQ = ac_smem(&b->fullQ), bAL = ac_smem(&b->fullAL), bE = ac_smem(&b->emptyA), bD = ac_smem(&b->itemdone);
  int* done = reinterpret_cast<int*>(A.sync + 1);
  const int NB = t3_nb(A), EPB = A.r * (F3_N / T3_EPL), ITH = 128 + EPB, totalH = (NB + 2 * A.lag) * ITH;
  const int nD = (int)(F3_N * F3_PLANE / 64), bpg = A.gs / A.r, slots = A.R * A.r;      // blocks per group; ring slots in spinors
  int* doneP = done; int* doneX = done + NB; int* doneE = done + 2 * NB; int* doneD = done + 3 * NB + A.G;
  uint32_t phE = 0, phD = 0;
  int i = 0;
#ifdef T3_TIMING
  unsigned long long pr_[4] = {0, 0, 0, 0};
  const long long tl0_ = clock64();
#endif
  T3_P0();
  for (;;) {
    const int s = atomicAdd(&A.sync->nextH, 1);
    if (s >= totalH) break;
    const int tick = s / ITH, q = s - tick * ITH, kind = q < 64 ? 0 : q < 128 ? 1 : 2, blk = tick - kind * A.lag;
    if (blk < 0 || blk >= NB) continue;
    if (kind == 0) { if (blk >= A.R) t3_wait(&doneE[blk - A.R], 2 * EPB, A.sync, A.spin_limit); }      // the QL slots have been read by E
    else if (kind == 1) t3_wait(&doneP[blk], 64, A.sync, A.spin_limit);                                // Q of the whole block is there
    else {
      t3_wait(&doneX[blk], 64, A.sync, A.spin_limit);                                                  // L of the whole block is there
      if (MODE != F3_APPLY && blk >= A.R) t3_wait(&doneD[(blk - A.R) / bpg], nD, A.sync, A.spin_limit);  // the X slots have been read by D
    }
    T3_P(0);
    const int n0 = blk * A.r;
    if (kind == 2) {                                            // E: no tiles, the pair reads global memory itself
      const int u = q - 128, k = u / (F3_N / T3_EPL), x0 = (u - k * (F3_N / T3_EPL)) * T3_EPL, n = n0 + k;
      if (n >= a.n) { f3_red_release(&doneE[blk]); f3_red_release(&doneE[blk]); continue; }
      const double sc = a.scale ? a.scale[n] : 1.0;
      for (int e = 0; e < T3_EPL; ++e, ++i) {
        T3_P(3);
        if (i > 0) { ac_mbar_wait(bE, phE); phE ^= 1; }
        T3_P(1);
        T3Mail* m = mail + (i & 1);
        m->kind = 2; m->n = n; m->c = 0; m->idx = x0 + e; m->slot = (n % slots) << 1; m->new_alpha = 0;
        m->done_idx = (e == T3_EPL - 1) ? 2 * NB + blk : -1;
        m->s = sc;
        ac_mbar_arrive(bA);
        T3_P(3);
        if (i > 0) { ac_mbar_wait(bD, phD); phD ^= 1; }
        T3_P(2);
      }
      continue;
    }
    ac_fence_proxy_global();                                    // ring data written by plain stores, read below by TMA
    const int u = q - kind * 64, c = u >> 5, idx = u & 31;
    int nvalid = a.n - n0; if (nvalid > A.r) nvalid = A.r;
    for (int k = 0; k < nvalid; ++k, ++i) {
      const int n = n0 + k, slot = ((n % slots) << 1) + c;
      T3_P(3);
      if (i > 0) { ac_mbar_wait(bE, phE); phE ^= 1; }
      T3_P(1);
      T3Mail* m = mail + (i & 1);
      m->kind = kind; m->n = n; m->c = c; m->idx = idx; m->slot = slot; m->new_alpha = (k == 0);
      m->done_idx = (k == nvalid - 1) ? kind * NB + blk : -1;
      m->s = a.scale ? a.scale[n] : 1.0;
      ac_mbar_expect_tx(bA, T3_TILE_BYTES);
      if (kind == 0) {
#pragma unroll
        for (int zg = 0; zg < 4; ++zg) t3_tma3(sA + zg * 4096, &maps.psiP, zg * 16, 0, ((n << 1) + c) * F3_N + idx, bA, pol.keep);
      } else {
        t3_tma4(sA, &maps.psiX, 0, idx, 0, (n << 1) + c, bA, pol.keep);
      }
      T3_P(3);
      if (i > 0) { ac_mbar_wait(bD, phD); phD ^= 1; }
      T3_P(2);
      if (k == 0) {
        ac_mbar_expect_tx(bAL, T3_AL_BYTES);
        if (kind == 0) {
#pragma unroll
          for (int zg = 0; zg < 2; ++zg) t3_tma4(sAL + zg * 4096, &maps.alP, zg * 16, 0, idx, c, bAL, pol.keep);
        } else {
          t3_tma4(sAL, &maps.alX, 0, idx, 0, c, bAL, pol.keep);
        }
      }
      if (kind == 1) {
        ac_mbar_expect_tx(bQ, T3_TILE_BYTES);
        t3_tma4(sB1, &maps.qlX, 0, idx, 0, slot, bQ, pol.keep);
      }
    }
  }
  if (i > 0) ac_mbar_wait(bE, phE);
  mail[i & 1].kind = -1;
  ac_mbar_arrive(bA);
#ifdef T3_TIMING
  atomicAdd(&g_t3_prof[0], pr_[0]); atomicAdd(&g_t3_prof[1], pr_[1]); atomicAdd(&g_t3_prof[2], pr_[2]);
  atomicAdd(&g_t3_prof[3], (unsigned long long)(clock64() - tl0_));
#endif
}

// ---- E: the pointwise epilogue of one (spinor, x-plane); warp t of the pair takes the rows y = 16 t .. 16 t + 15 in
// four batches of four rows (lane = z): all 32 loads of a batch are in flight before the first use (the line registers
// are free between transforms).  K_c = -L_c / 4 (+ (lap alpha_c) w / 4 inside q, + the transverse shift), the BdG mix,
// the eps_n / norm partial sums and the stage combination; the warp that completes a spinor turns the partial sums into
// eps_n and 1 / |phi_new|. ---------------------------------------------------------------------------------------------
template <int MODE>
__device__ __forceinline__ void t3_body_e(const T3Mega& A, const F3Pol& pol, const T3Mail& m, int t, int lane, cplx* x) {
  const F3Mega& a = A.m;
  const int n = m.n, ix = m.idx;
  const size_t M = (size_t)F3_N * F3_PLANE, off = (size_t)ix * F3_PLANE + (size_t)(16 * t) * F3_N + lane;
  const double s = m.s, kp2 = a.kperp2[n];
  const cplx* pu = a.psi + (size_t)(2 * n) * M + off;
  const cplx* pk = a.pack + off;
  const cplx* Lu = a.spec0 + (size_t)m.slot * M + off;
  const cplx* cu = a.cpart + (size_t)(2 * n) * M + off;
  cplx* ou = (MODE == F3_APPLY ? a.out + (size_t)(2 * n) * M : a.X + (size_t)m.slot * M) + off;
  double e = 0.0, xx = 0.0, xpr = 0.0, xpi = 0.0, pp = 0.0;
#pragma unroll 1
  for (int b = 0; b < 4; ++b) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const size_t i = (size_t)(4 * b + r) * F3_N;
      x[8 * r + 0] = pu[i]; x[8 * r + 1] = pu[M + i];
      x[8 * r + 2] = ld_pol(Lu + i, pol.drop); x[8 * r + 3] = ld_pol(Lu + M + i, pol.drop);       // last use of L
      x[8 * r + 4] = pk[i]; x[8 * r + 5] = pk[M + i];
      if (MODE == F3_CORR) { x[8 * r + 6] = ld_pol(cu + i, pol.drop); x[8 * r + 7] = ld_pol(cu + M + i, pol.drop); }   // read once
    }
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const size_t i = (size_t)(4 * b + r) * F3_N;
      const cplx u = cscale(x[8 * r + 0], s), v = cscale(x[8 * r + 1], s);
      const cplx lu = x[8 * r + 2], lv = x[8 * r + 3], q = x[8 * r + 4], D = x[8 * r + 5];
      double ha = 0.5 * kp2, hb = 0.5 * kp2;
      if (kp2 != 0.0) { const cplx al = pk[2 * M + i]; ha *= al.x; hb *= al.y; }
      const cplx Ku = make_double2(-0.25 * lu.x + ha * u.x, -0.25 * lu.y + ha * u.y);    // Eq. 40 (its +(lap alpha) w / 4 sits in q)
      const cplx Kv = make_double2(-0.25 * lv.x + hb * v.x, -0.25 * lv.y + hb * v.y);
      const cplx Hu = cadd(Ku, cadd(cscale(u, q.x), cmul(D, v)));                        // Eqs. 5, 15
      const cplx Hv = csub(cmul(cconj(D), u), cadd(Kv, cscale(v, q.y)));
      e += u.x * Hu.x + u.y * Hu.y + v.x * Hv.x + v.y * Hv.y;
      if (MODE == F3_APPLY) { st_pol_nb(ou + i, Hu, pol.drop); st_pol_nb(ou + M + i, Hv, pol.drop); }
      else if (MODE == F3_RHS) {                                                          // -i H
        st_pol_nb(ou + i, make_double2(Hu.y, -Hu.x), pol.keep); st_pol_nb(ou + M + i, make_double2(Hv.y, -Hv.x), pol.keep);
      } else {
        const cplx c0 = x[8 * r + 6], c1 = x[8 * r + 7];
        const cplx xu = make_double2(c0.x + a.kappa * Hu.y, c0.y - a.kappa * Hu.x);       // C_part - i kappa H
        const cplx xv = make_double2(c1.x + a.kappa * Hv.y, c1.y - a.kappa * Hv.x);
        st_pol_nb(ou + i, xu, pol.keep); st_pol_nb(ou + M + i, xv, pol.keep);
        xx += cabs2(xu) + cabs2(xv);
        xpr += xu.x * u.x + xu.y * u.y + xv.x * v.x + xv.y * v.y;
        xpi += xu.x * u.y - xu.y * u.x + xv.x * v.y - xv.y * v.x;
        pp += cabs2(u) + cabs2(v);
      }
    }
  }
  e = warp_sum(e);
  if (MODE == F3_CORR) { xx = warp_sum(xx); xpr = warp_sum(xpr); xpi = warp_sum(xpi); pp = warp_sum(pp); }
  const size_t np = (size_t)a.n * 64, o = (size_t)n * 64 + 2 * ix + t;
  if (lane == 0) {
    a.part[o] = e;
    if (MODE == F3_CORR) { a.part[np + o] = xx; a.part[2 * np + o] = xpr; a.part[3 * np + o] = xpi; a.part[4 * np + o] = pp; }
  }
}

// ---- S: the scalars of one spinor from its 64 partial sums (one light warp, fixed order): eps_n = Re dV sum psi^+ H psi
// (Eq. 44b) and, for the corrector, 1 / |X + i kappa eps w| (Alg. 2 step 8; R26) ----------------------------------------
template <int MODE>
__device__ __forceinline__ void t3_body_s(const T3Mega& A, int n, int lane) {
  const F3Mega& a = A.m;
  if (n >= a.n) return;
  const size_t np = (size_t)a.n * 64;
  double v[F3_NPART];
#pragma unroll
  for (int k = 0; k < F3_NPART; ++k) {
    v[k] = 0.0;
    if (k == 0 || MODE == F3_CORR) {
      const double* pp_ = a.part + k * np + (size_t)n * 64;
      v[k] = warp_sum(__ldcg(pp_ + lane) + __ldcg(pp_ + 32 + lane));
    }
  }
  if (lane == 0) {
    const double e_true = a.dV * v[0];
    if (a.eps_out) a.eps_out[n] = e_true;
    if (MODE == F3_APPLY && A.eps_user) A.eps_user[n] = e_true;
    if (MODE == F3_CORR) {
      const double ke = a.kappa * (a.use_shift ? e_true : 0.0), nrm2 = a.dV * (v[1] - 2.0 * ke * v[3] + ke * ke * v[4]);
      A.sn_out[n] = a.normalize ? 1.0 / sqrt(nrm2) : 1.0;
    }
  }
}

// the two heavy warps of pair `pr`
template <int MODE>
__device__ __forceinline__ void t3_heavy(const T3Mega& A, unsigned char* smem, int pr, int t, int lane
#ifdef T3_TIMING
                                         , unsigned long long* cyc
#endif
) {
  const F3Mega& a = A.m;
  const F3Pol pol = f3_policies();
  cplx x[F3_N];
  T3Pair p;
  p.base = smem + pr * T3_PAIR_BYTES; p.bars = reinterpret_cast<T3Bars*>(smem + T3_MISC_OFF) + pr;
  p.phA = p.phQ = p.phAL = p.phH = p.phF = p.phM = 0;
  p.t = t; p.lane = lane;
#ifdef T3_TIMING
  p.cyc = cyc;
#endif
  const T3Mail* mail = reinterpret_cast<const T3Mail*>(smem + T3_MISC_OFF + T3_PAIRS * sizeof(T3Bars)) + pr * 2;
  int* done = reinterpret_cast<int*>(A.sync + 1);
  const size_t M = (size_t)F3_N * F3_PLANE;
  for (int i = 0;; ++i) {
#ifdef T3_TIMING
    long long t_ = clock64();
#endif
    ac_mbar_wait(ac_smem(&p.bars->fullA), p.phA); p.phA ^= 1;
    const T3Mail m = mail[i & 1];
    if (m.kind < 0) break;
    if (m.kind == 2) {                                          // E: no tiles
      if (lane == 0) ac_mbar_arrive(ac_smem(&p.bars->emptyA));
      T3_T(0, 1);
      t3_body_e<MODE>(A, pol, m, t, lane, x);
      __syncwarp();
      if (lane == 0) { if (m.done_idx >= 0) f3_red_release(&done[m.done_idx]); ac_mbar_arrive(ac_smem(&p.bars->itemdone)); }
      T3_T(0, 3);
      continue;
    }
    if (m.new_alpha) { ac_mbar_wait(ac_smem(&p.bars->fullAL), p.phAL); p.phAL ^= 1; }
    T3_T(m.kind, 1);
    cplx* ring = a.spec0 + (size_t)m.slot * M;
    t3_body_px(p, m.kind, ring + (size_t)m.idx * (m.kind ? F3_N : F3_PLANE), m.s, A.k2all, pol, x);
    if (m.done_idx >= 0 && t == m.kind) {                       // this warp made the item's global stores
      ac_fence_proxy_global();
      __syncwarp();
      if (lane == 0) f3_red_release(&done[m.done_idx]);
    }
    __syncwarp();
    if (lane == 0) ac_mbar_arrive(ac_smem(&p.bars->itemdone));
  }
}

// ---- D: the closing combination of 64 lattice points (two per lane) for every spinor of a group, by one light warp ----
// CORR: phi_new = (X + i kappa eps w) / |.| over P (Alg. 2 steps 4, 8) + densities of phi_new into the group's ring slot;
// RHS : f_new = Y + i eps phi (Alg. 2 step 9, Eq. 45b).
#define T3_DPTS 64
template <int MODE>
__device__ __forceinline__ void t3_body_d(const T3Mega& A, const F3Pol& pol, int g, int id, int lane) {
  const F3Mega& a = A.m;
  const int cnt = (a.n - g * A.gs < A.gs) ? a.n - g * A.gs : A.gs;
  const size_t M = (size_t)F3_N * F3_PLANE, p0 = (size_t)id * T3_DPTS + lane;
  const int slots = A.R * A.r;
  double acc[2][4];
#pragma unroll
  for (int r = 0; r < 2; ++r) { acc[r][0] = acc[r][1] = acc[r][2] = acc[r][3] = 0.0; }
#pragma unroll 1
  for (int nl = 0; nl < cnt; ++nl) {
    const int n = g * A.gs + nl;
    const cplx* Xu = a.X + (size_t)((n % slots) * 2) * M + p0;
    const cplx* pu = a.psi + (size_t)(2 * n) * M + p0;
    cplx* ou = a.out + (size_t)(2 * n) * M + p0;
    cplx gxu[2], gxv[2], gpu[2], gpv[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) { gxu[r] = __ldcg(Xu + r * 32); gxv[r] = __ldcg(Xu + M + r * 32); gpu[r] = pu[r * 32]; gpv[r] = pu[M + r * 32]; }
    const double e = a.use_shift ? __ldcg(a.eps_out + n) : 0.0;
    if (MODE == F3_CORR) {
      const double sP = a.scale ? a.scale[n] : 1.0, ke = a.kappa * e, sn = __ldcg(A.sn_out + n);
      const double cp = a.cpref[n], wa = a.w_a[n], wb = a.w_b[n];
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        const cplx wu = cscale(gpu[r], sP), wv = cscale(gpv[r], sP);
        const cplx u = make_double2((gxu[r].x - ke * wu.y) * sn, (gxu[r].y + ke * wu.x) * sn);
        const cplx v = make_double2((gxv[r].x - ke * wv.y) * sn, (gxv[r].y + ke * wv.x) * sn);
        st_pol_nb(ou + r * 32, u, pol.drop); st_pol_nb(ou + M + r * 32, v, pol.drop);
        if (a.do_dens) f3_dens_add(acc[r], u, v, cp, wa, wb);
      }
    } else {
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        st_pol_nb(ou + r * 32, make_double2(gxu[r].x - e * gpu[r].y, gxu[r].y + e * gpu[r].x), pol.drop);
        st_pol_nb(ou + M + r * 32, make_double2(gxv[r].x - e * gpv[r].y, gxv[r].y + e * gpv[r].x), pol.drop);
      }
    }
  }
  if (MODE == F3_CORR && a.do_dens) {
    double* ac = a.acc + (size_t)(g % A.RA) * 4 * M + p0;
#pragma unroll
    for (int r = 0; r < 2; ++r)
#pragma unroll
      for (int f = 0; f < 4; ++f) {
        double* q = ac + f * M + r * 32;
        *q = (g < A.RA ? 0.0 : __ldcg(q)) + acc[r][f];
      }
  }
}

// a light warp: draws the light tickets; per group g: S(g) [gs items, one spinor each], then D(g) [M / 64 items]
template <int MODE>
__device__ __forceinline__ void t3_light(const T3Mega& A, int lane) {
  const F3Pol pol = f3_policies();
  int* done = reinterpret_cast<int*>(A.sync + 1);
  const int G = A.G, NB = t3_nb(A), EPB = A.r * (F3_N / T3_EPL), nD = MODE == F3_APPLY ? 0 : (int)(F3_N * F3_PLANE / T3_DPTS);
  int* doneE = done + 2 * NB; int* doneS = done + 3 * NB; int* doneD = done + 3 * NB + G;
  const int ITL = A.gs + nD, totalL = G * ITL;
#ifdef T3_TIMING
  unsigned long long pr_[12] = {0};
  const long long tl0_ = clock64();
#endif
  T3_P0();
  for (;;) {
    int s = 0;
    if (lane == 0) s = atomicAdd(&A.sync->nextL, 1);
    s = __shfl_sync(0xffffffffu, s, 0);
    T3_P(10);
    if (s >= totalL) break;
    const int g = s / ITL, q = s - g * ITL;
    if (q < A.gs) {                                             // S: every E item of the spinor's block has left its partial sums
      const int n = g * A.gs + q;
      if (lane == 0 && n < A.m.n) t3_wait(&doneE[n / A.r], 2 * EPB, A.sync, A.spin_limit);
      __syncwarp();
      T3_P(6);
      t3_body_s<MODE>(A, n, lane);
      T3_P(7);
      __syncwarp();
      if (lane == 0) f3_red_release(&doneS[g]);
      continue;
    }
    if (lane == 0) {
      t3_wait(&doneS[g], A.gs, A.sync, A.spin_limit);                                             // X, eps_n, |phi_new| of the group are complete
      if (g >= A.RA) t3_wait(&doneD[g - A.RA], nD, A.sync, A.spin_limit);                           // the density slot
    }
    __syncwarp();
    T3_P(6);
    t3_body_d<MODE>(A, pol, g, q - A.gs, lane);
    T3_P(8);
    __syncwarp();
    if (lane == 0) f3_red_release(&doneD[g]);
  }
#ifdef T3_TIMING
  if (lane == 0) {
    atomicAdd(&g_t3_prof[6], pr_[6]); atomicAdd(&g_t3_prof[7], pr_[7]); atomicAdd(&g_t3_prof[8], pr_[8]); atomicAdd(&g_t3_prof[10], pr_[10]);
    atomicAdd(&g_t3_prof[9], (unsigned long long)(clock64() - tl0_));
  }
#endif
}

template <int MODE>
__global__ void __launch_bounds__(T3_THREADS, 1) k_t3_mega(const __grid_constant__ T3Maps maps, const __grid_constant__ T3Mega A) {
  extern __shared__ __align__(1024) unsigned char t3_smem[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    T3Bars* bars = reinterpret_cast<T3Bars*>(t3_smem + T3_MISC_OFF);
    for (int i = 0; i < T3_PAIRS; ++i) {
      ac_mbar_init(ac_smem(&bars[i].fullA), 1); ac_mbar_init(ac_smem(&bars[i].fullQ), 1); ac_mbar_init(ac_smem(&bars[i].fullAL), 1);
      ac_mbar_init(ac_smem(&bars[i].emptyA), 2); ac_mbar_init(ac_smem(&bars[i].itemdone), 2);
      ac_mbar_init(ac_smem(&bars[i].hready), 1); ac_mbar_init(ac_smem(&bars[i].hfree), 1); ac_mbar_init(ac_smem(&bars[i].mail), 1);
    }
    ac_fence_mbar_init();
  }
#ifdef T3_TIMING
  __shared__ unsigned long long s_cyc[8][16];
  if (threadIdx.x < 128) s_cyc[threadIdx.x >> 4][threadIdx.x & 15] = 0;
#endif
  __syncthreads();
  if (warp >= 2 * T3_PAIRS) {
    ac_reg_dec<T3_LIGHT_REGS>();
    if (warp == 2 * T3_PAIRS) { if (lane < T3_PAIRS) t3_loader<MODE>(maps, A, t3_smem, lane); }
    else t3_light<MODE>(A, lane);
    return;
  }
  ac_reg_inc<T3_HEAVY_REGS>();
#ifdef T3_TIMING
  const long long th0_ = clock64();
  t3_heavy<MODE>(A, t3_smem, warp >> 1, warp & 1, lane, s_cyc[warp]);
  __syncwarp();
  if (lane < 16) atomicAdd(&g_t3_cycles[warp & 1][lane], s_cyc[warp][lane]);
  if (lane == 0) atomicAdd(&g_t3_prof[5], (unsigned long long)(clock64() - th0_));
#else
  t3_heavy<MODE>(A, t3_smem, warp >> 1, warp & 1, lane);
#endif
}

#ifdef T3_TIMING
extern "C" void wslda_debug_t3_cycles(unsigned long long* heavy32, unsigned long long* prof16) {
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(heavy32, g_t3_cycles, sizeof(unsigned long long) * 32);
  cudaMemcpyFromSymbol(prof16, g_t3_prof, sizeof(unsigned long long) * 16);
  unsigned long long z[32] = {0};
  cudaMemcpyToSymbol(g_t3_cycles, z, sizeof(unsigned long long) * 32); cudaMemcpyToSymbol(g_t3_prof, z, sizeof(unsigned long long) * 16);
}
#endif
