// fft_radix.cuh — small complex DFTs held entirely in registers (fp64), the butterflies of the xy FFT passes (fft.cu).
//
//   Dft<R, INV>::run(x)   x[k] <- sum_n x[n] W^{nk},  W = exp(-2 pi i / R)  (INV: exp(+2 pi i / R)), unnormalised,
//   for R in {2, 3, 4, 5, 8, 9, 15, 16, 18}.  Primes and 4 are written out; 8 = 2x4, 9 = 3x3 and 16 = 4x4 are
//   Cooley-Tukey products with constant twiddles; 15 = 3x5 and 18 = 2x9 use the Good-Thomas index maps (coprime
//   factors, no twiddles).  Everything is fully unrolled: array indices are compile-time after unrolling, so the
//   arrays live in registers and the twiddle constants become immediate operands.
//   The functions are __host__ __device__ so that the index logic can be checked on the CPU.
#pragma once

#include <cuda_runtime.h>

#define DP_HD __host__ __device__ __forceinline__

namespace dpfft {

DP_HD double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
DP_HD double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
// a * (c - i s)  (forward twiddle stored as (c, -s): pass w = (c, -s) and use cmul)
DP_HD double2 cmul(double2 a, double2 w) { return make_double2(fma(a.x, w.x, -a.y * w.y), fma(a.x, w.y, a.y * w.x)); }
// a * conj(w)
DP_HD double2 cmulc(double2 a, double2 w) { return make_double2(fma(a.x, w.x, a.y * w.y), fma(a.y, w.x, -a.x * w.y)); }
// a * (-i) forward, a * (+i) inverse
template <bool INV> DP_HD double2 mul_mi(double2 a) { return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x); }

// cos(2 pi j / R), sin(2 pi j / R) for the composite radices with internal twiddles (R = 8, 9, 16)
DP_HD constexpr double tw_cos16(int j) {
  return j == 0 ? 1.0 : j == 1 ? 0.92387953251128675613 : j == 2 ? 0.70710678118654752440 : j == 3 ? 0.38268343236508977173
       : j == 4 ? 0.0 : j == 5 ? -0.38268343236508977173 : j == 6 ? -0.70710678118654752440 : j == 7 ? -0.92387953251128675613
       : j == 8 ? -1.0 : j == 9 ? -0.92387953251128675613 : j == 10 ? -0.70710678118654752440 : j == 11 ? -0.38268343236508977173
       : j == 12 ? 0.0 : j == 13 ? 0.38268343236508977173 : j == 14 ? 0.70710678118654752440 : 0.92387953251128675613;
}
DP_HD constexpr double tw_sin16(int j) { return tw_cos16((j + 12) & 15); }      // sin(t) = cos(t - pi/2)
DP_HD constexpr double tw_cos9(int j) {
  return j == 0 ? 1.0 : (j == 1 || j == 8) ? 0.76604444311897803520 : (j == 2 || j == 7) ? 0.17364817766693034885
       : (j == 3 || j == 6) ? -0.5 : -0.93969262078590838405;
}
DP_HD constexpr double tw_sin9(int j) {
  return j == 0 ? 0.0 : j == 1 ? 0.64278760968653932632 : j == 2 ? 0.98480775301220805937 : j == 3 ? 0.86602540378443864676
       : j == 4 ? 0.34202014332566873304 : j == 5 ? -0.34202014332566873304 : j == 6 ? -0.86602540378443864676
       : j == 7 ? -0.98480775301220805937 : -0.64278760968653932632;
}

// a * W_R^j with W_R = exp(-+ 2 pi i / R); j is a compile-time value after unrolling, so the branches fold
template <int R, bool INV> DP_HD double2 mul_tw(double2 a, int j) {
  j %= R;
  if (j == 0) return a;
  if (4 * j == R) return mul_mi<INV>(a);
  if (2 * j == R) return make_double2(-a.x, -a.y);
  if (4 * j == 3 * R) return mul_mi<!INV>(a);
  const double c = (R == 9) ? tw_cos9(j) : tw_cos16(j * (16 / (R == 9 ? 16 : R)));
  const double s = (R == 9) ? tw_sin9(j) : tw_sin16(j * (16 / (R == 9 ? 16 : R)));
  const double2 w = make_double2(c, INV ? s : -s);
  return cmul(a, w);
}

template <int R, bool INV> struct Dft;

template <bool INV> struct Dft<2, INV> {
  static DP_HD void run(double2 (&x)[2]) {
    const double2 a = x[0], b = x[1];
    x[0] = cadd(a, b); x[1] = csub(a, b);
  }
};

template <bool INV> struct Dft<3, INV> {
  static DP_HD void run(double2 (&x)[3]) {
    constexpr double S3 = 0.86602540378443864676;
    const double2 s = cadd(x[1], x[2]), d = csub(x[1], x[2]);
    const double2 m = make_double2(fma(-0.5, s.x, x[0].x), fma(-0.5, s.y, x[0].y));
    x[0] = cadd(x[0], s);
    const double2 q = mul_mi<INV>(make_double2(S3 * d.x, S3 * d.y));     // -+ i S3 d
    x[1] = cadd(m, q); x[2] = csub(m, q);
  }
};

template <bool INV> struct Dft<4, INV> {
  static DP_HD void run(double2 (&x)[4]) {
    const double2 a = cadd(x[0], x[2]), b = csub(x[0], x[2]), c = cadd(x[1], x[3]), d = mul_mi<INV>(csub(x[1], x[3]));
    x[0] = cadd(a, c); x[2] = csub(a, c); x[1] = cadd(b, d); x[3] = csub(b, d);
  }
};

template <bool INV> struct Dft<5, INV> {
  static DP_HD void run(double2 (&x)[5]) {
    constexpr double C1 = 0.30901699437494742410, C2 = -0.80901699437494742410;
    constexpr double S1 = 0.95105651629515357212, S2 = 0.58778525229247312917;
    const double2 a1 = cadd(x[1], x[4]), a2 = cadd(x[2], x[3]), b1 = csub(x[1], x[4]), b2 = csub(x[2], x[3]);
    const double2 m1 = make_double2(fma(C1, a1.x, fma(C2, a2.x, x[0].x)), fma(C1, a1.y, fma(C2, a2.y, x[0].y)));
    const double2 m2 = make_double2(fma(C2, a1.x, fma(C1, a2.x, x[0].x)), fma(C2, a1.y, fma(C1, a2.y, x[0].y)));
    const double2 n1 = mul_mi<INV>(make_double2(fma(S1, b1.x, S2 * b2.x), fma(S1, b1.y, S2 * b2.y)));
    const double2 n2 = mul_mi<INV>(make_double2(fma(S2, b1.x, -S1 * b2.x), fma(S2, b1.y, -S1 * b2.y)));
    x[0] = cadd(x[0], cadd(a1, a2));
    x[1] = cadd(m1, n1); x[4] = csub(m1, n1); x[2] = cadd(m2, n2); x[3] = csub(m2, n2);
  }
};

// Cooley-Tukey R = R1 R2: n = R2 n1 + n2, k = k1 + R1 k2
template <int R1, int R2, bool INV> DP_HD void dft_ct(double2 (&x)[R1 * R2]) {
  constexpr int R = R1 * R2;
  double2 y[R];
#pragma unroll
  for (int n2 = 0; n2 < R2; ++n2) {
    double2 t[R1];
#pragma unroll
    for (int n1 = 0; n1 < R1; ++n1) t[n1] = x[R2 * n1 + n2];
    Dft<R1, INV>::run(t);
#pragma unroll
    for (int k1 = 0; k1 < R1; ++k1) y[k1 * R2 + n2] = mul_tw<R, INV>(t[k1], k1 * n2);
  }
#pragma unroll
  for (int k1 = 0; k1 < R1; ++k1) {
    double2 u[R2];
#pragma unroll
    for (int n2 = 0; n2 < R2; ++n2) u[n2] = y[k1 * R2 + n2];
    Dft<R2, INV>::run(u);
#pragma unroll
    for (int k2 = 0; k2 < R2; ++k2) x[k1 + R1 * k2] = u[k2];
  }
}

// Good-Thomas R = R1 R2, gcd(R1, R2) = 1: n = (R2 n1 + R1 n2) mod R, k = (R2 U k1 + R1 V k2) mod R with
// U = R2^{-1} mod R1, V = R1^{-1} mod R2 (Chinese remainder theorem); no twiddles
template <int R1, int R2, int U, int V, bool INV> DP_HD void dft_pfa(double2 (&x)[R1 * R2]) {
  constexpr int R = R1 * R2;
  static_assert((R2 * U) % R1 == 1 % R1 && (R1 * V) % R2 == 1 % R2, "CRT inverses");
  double2 y[R];
#pragma unroll
  for (int n2 = 0; n2 < R2; ++n2) {
    double2 t[R1];
#pragma unroll
    for (int n1 = 0; n1 < R1; ++n1) t[n1] = x[(R2 * n1 + R1 * n2) % R];
    Dft<R1, INV>::run(t);
#pragma unroll
    for (int k1 = 0; k1 < R1; ++k1) y[k1 * R2 + n2] = t[k1];
  }
#pragma unroll
  for (int k1 = 0; k1 < R1; ++k1) {
    double2 u[R2];
#pragma unroll
    for (int n2 = 0; n2 < R2; ++n2) u[n2] = y[k1 * R2 + n2];
    Dft<R2, INV>::run(u);
#pragma unroll
    for (int k2 = 0; k2 < R2; ++k2) x[(R2 * U * k1 + R1 * V * k2) % R] = u[k2];
  }
}

template <bool INV> struct Dft<8, INV> { static DP_HD void run(double2 (&x)[8]) { dft_ct<2, 4, INV>(x); } };
template <bool INV> struct Dft<9, INV> { static DP_HD void run(double2 (&x)[9]) { dft_ct<3, 3, INV>(x); } };
template <bool INV> struct Dft<16, INV> { static DP_HD void run(double2 (&x)[16]) { dft_ct<4, 4, INV>(x); } };
template <bool INV> struct Dft<15, INV> { static DP_HD void run(double2 (&x)[15]) { dft_pfa<3, 5, 2, 2, INV>(x); } };   // 5*2 = 10 = 1 mod 3 ; 3*2 = 6 = 1 mod 5
template <bool INV> struct Dft<18, INV> { static DP_HD void run(double2 (&x)[18]) { dft_pfa<2, 9, 1, 5, INV>(x); } };   // 9*1 = 1 mod 2 ; 2*5 = 10 = 1 mod 9

}  // namespace dpfft
