// regfft.cuh -- register-resident complex128 FFTs of length 2..32 (one lattice line per thread).
// Every index is a compile-time constant after unrolling, so the line lives in registers and the twiddles
// are immediates; the transform is the plain DFT of Eq. 26: forward sum_r x_r e^{-2 pi i k r/N},
// inverse with e^{+...} and no normalisation (the 1/M is folded into the k-space factor).
// Decimation in frequency, radix 2, in place; the bit-reversed result is renamed back to natural order.
#pragma once
#include "common.cuh"

// cos(2 pi k / 64), k = 0..16, correctly rounded; the other quadrants follow by symmetry so that the table is
// exactly symmetric.
__host__ __device__ constexpr double ws_cos64_q(int k) {
  switch (k) {
    case 0: return 1.0;
    case 1: return 0.99518472667219688624;
    case 2: return 0.98078528040323044913;
    case 3: return 0.95694033573220886494;
    case 4: return 0.92387953251128675613;
    case 5: return 0.88192126434835502971;
    case 6: return 0.83146961230254523708;
    case 7: return 0.77301045336273696081;
    case 8: return 0.70710678118654752440;
    case 9: return 0.63439328416364549822;
    case 10: return 0.55557023301960222474;
    case 11: return 0.47139673682599764856;
    case 12: return 0.38268343236508977173;
    case 13: return 0.29028467725446236764;
    case 14: return 0.19509032201612826785;
    case 15: return 0.09801714032956060199;
    default: return 0.0;
  }
}
__host__ __device__ constexpr double ws_cos64(int k) {        // k in [0, 64)
  return k <= 16 ? ws_cos64_q(k) : k <= 32 ? -ws_cos64_q(32 - k) : k <= 48 ? -ws_cos64_q(k - 32) : ws_cos64_q(64 - k);
}
__host__ __device__ constexpr double ws_sin64(int k) { return ws_cos64((k + 48) & 63); }   // sin x = cos(x - pi/2)

__host__ __device__ constexpr int ws_brev(int i, int n) {
  int r = 0;
  for (int b = 1; b < n; b <<= 1) { r = (r << 1) | (i & 1); i >>= 1; }
  return r;
}

// d * exp(-/+ 2 pi i T / 64), T in [0, 32) a compile-time constant
template <int T, bool INV>
__device__ __forceinline__ cplx mul_tw64(cplx d) {
  if (T == 0) return d;
  if (T == 16) return INV ? make_double2(-d.y, d.x) : make_double2(d.y, -d.x);
  constexpr double c = ws_cos64(T), s = INV ? -ws_sin64(T) : ws_sin64(T);     // w = c - i s
  return make_double2(fma(d.y, s, d.x * c), fma(-d.x, s, d.y * c));
}

template <int N, int L, int B, int J, bool INV>
struct RegFftStage {
  static __device__ __forceinline__ void run(cplx* x) {
    constexpr int h = L / 2;
    const cplx a = x[B + J], c = x[B + J + h];
    x[B + J] = cadd(a, c);
    x[B + J + h] = mul_tw64<J * (64 / L), INV>(csub(a, c));
    if constexpr (J + 1 < h) RegFftStage<N, L, B, J + 1, INV>::run(x);
    else if constexpr (B + L < N) RegFftStage<N, L, B + L, 0, INV>::run(x);
    else if constexpr (L > 2) RegFftStage<N, L / 2, 0, 0, INV>::run(x);
  }
};

template <int N, int I>
struct RegFftPermute {
  static __device__ __forceinline__ void run(cplx* x) {
    constexpr int r = ws_brev(I, N);
    if constexpr (r > I) { const cplx t = x[I]; x[I] = x[r]; x[r] = t; }
    if constexpr (I + 1 < N) RegFftPermute<N, I + 1>::run(x);
  }
};

// in-place transform of x[0..N), natural order in and out; N in {2, 4, 8, 16, 32, 64}
template <int N, bool INV>
__device__ __forceinline__ void fft_reg(cplx* x) {
  static_assert(N >= 2 && N <= 64 && (N & (N - 1)) == 0, "line length");
  RegFftStage<N, N, 0, 0, INV>::run(x);
  RegFftPermute<N, 0>::run(x);
}
