// solve_common.cuh — pieces shared by the two per-wavenumber solve kernels (solve.cu: tile kernel with the Fourier-curl torque
// fields; solve_pair.cu: register-resident warp-pair kernel for three fields each way): launch arguments, the tridiagonal rows of
// the integration-form BVP chains, the wall-correction coefficients (eqs 42-44; App. A) and the 4x4 solve of the slit.
#pragma once

#include "common.cuh"

namespace dp_solve {

constexpr int TM = DP_SOLVE_TM;        // modes per CTA
constexpr int LN = 2 * TM;             // lanes of a complex column row (= 32)
static_assert(LN == 32, "a warp row is one complex column row");

struct SolveArgs {
  double2* cplx;
  size_t cplx_field;
  int nx, ny, nkx;
  int n_fast, n_slow, pitch;     // half spectrum stored as [field][l][slow][fast (pitch)]
  int fast_is_x;                 // 1: fast index = kx index (cuFFT layout); 0: fast index = position along ky (transposed layout)
  const int* lmin;               // planes l < *lmin of the input hold zeros that were never written: not read
  const int* ky_of_pos;          // transposed layout: FFT-order ky index stored at each position (digit reversal of the y pass), or null
  const double* frag;            // transform fragment table (see Tr)
  double Lx, Ly, H, eta;
  int wall_mode, torque, omega;
  int slip;                      // slit with a non-zero slip length (App. A)
  double l0, lH;                 // slip lengths of the bottom / top wall
  double uw0[2], uwH[2];         // uniform wall velocities (x, y): enter the k = 0 column only
};

__device__ __forceinline__ void cp_async16(double* smem_dst, const double2* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ double ldg_stream(const double* p) {
  double v;
  asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void named_sync(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
__device__ __forceinline__ void named_arrive(int id, int nthreads) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }

// ---- branch-free 1/x and e^x (x <= 0).  The library routines guard their special cases with a branch to a slow path; in code that is
// one long basic block per phase every such branch costs an instruction-fetch bubble (BSSY / BSYNC), and the operands here are
// well-conditioned pivots, wavenumbers and exponents, never zero, infinite or denormal.
__device__ __forceinline__ double dp_rcp(double d) {          // two Newton steps on the hardware seed: <= 1 ulp
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
  double e = fma(-d, r, 1.0);
  r = fma(r, e, r);
  e = fma(-d, r, 1.0);
  return fma(r, e, r);
}
__device__ __forceinline__ double dp_exp_neg(double x) {      // e^x for x <= 0 (x < -700 gives e^-700: the terms it scales are then < 1e-300 of the rest)
  x = fmax(x, -700.0);
  const double t = rint(x * 1.4426950408889634074);
  double r = fma(t, -6.93147180369123816490e-01, x);          // x - t ln 2, ln 2 split in two
  r = fma(t, -1.90821492927058770002e-10, r);
  // |r| <= 0.3466: Taylor polynomial of degree 13, remainder < 5e-18
  double p = 1.6059043836821613e-10;                          // 1/13!
  p = fma(p, r, 2.08767569878681e-09);                        // 1/12!
  p = fma(p, r, 2.505210838544172e-08);
  p = fma(p, r, 2.755731922398589e-07);
  p = fma(p, r, 2.755731922398589e-06);
  p = fma(p, r, 2.48015873015873e-05);
  p = fma(p, r, 1.984126984126984e-04);
  p = fma(p, r, 1.388888888888889e-03);
  p = fma(p, r, 8.333333333333333e-03);
  p = fma(p, r, 4.1666666666666664e-02);
  p = fma(p, r, 1.6666666666666666e-01);
  p = fma(p, r, 0.5);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  return p * __hiloint2double((1023 + (int)t) << 20, 0);      // 2^t, t in [-1010, 0]
}

// the same with the Taylor coefficients 1/13!, ..., 1/2! read from a table `ec` (a kernel-parameter array: one uniform load per coefficient
// instead of two immediate moves)
__device__ __forceinline__ double dp_exp_neg_tab(double x, const double (&ec)[12]) {
  x = fmax(x, -700.0);
  const double t = rint(x * 1.4426950408889634074);
  double r = fma(t, -6.93147180369123816490e-01, x);
  r = fma(t, -1.90821492927058770002e-10, r);
  double p = ec[0];
#pragma unroll
  for (int q = 1; q < 12; ++q) p = fma(p, r, ec[q]);
  p = fma(p, r, 1.0);
  p = fma(p, r, 1.0);
  return p * __hiloint2double((1023 + (int)t) << 20, 0);
}

// ---- tridiagonal rows of a chain (n >= 1): d_n a_n + l_n a_{n-2} + u_n a_{n+2}; all divisions are compile-time constants
template <int NZ> __device__ __forceinline__ double row_d(int n, double k2) { return n == 1 ? fma(k2, 0.125, 1.0) : fma(k2, 1.0 / (2.0 * (n * n - 1)), 1.0); }
template <int NZ> __device__ __forceinline__ double row_l(int n, double k2) { return k2 * (-(n == 2 ? 2.0 : 1.0) / (4.0 * n * (n - 1))); }
template <int NZ> __device__ __forceinline__ double row_u(int n, double k2) { return (n + 2 <= NZ - 3) ? k2 * (-1.0 / (4.0 * n * (n + 1))) : 0.0; }

// ---- chain geometry: rows n0, n0+2, ... <= N-2 of parity PAR
template <int NZ, int PAR> struct Ch {
  static constexpr int N = NZ - 1, n0 = PAR ? 1 : 2, NR = PAR ? (N - 1) / 2 : (N - 2) / 2;
};

// ---- 4x4 real system, one right-hand side per lane, partial pivoting after row equilibration
__device__ __forceinline__ void solve4(double M[4][4], double b[4]) {
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const double mx = fmax(fmax(fabs(M[r][0]), fabs(M[r][1])), fmax(fabs(M[r][2]), fabs(M[r][3])));
    const double s = mx > 0.0 ? dp_rcp(mx) : 1.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) M[r][c] *= s;
    b[r] *= s;
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) {
#pragma unroll
    for (int r = c + 1; r < 4; ++r) {                       // bubble the largest pivot candidate into row c
      if (fabs(M[r][c]) > fabs(M[c][c])) {
#pragma unroll
        for (int q = 0; q < 4; ++q) { const double t = M[c][q]; M[c][q] = M[r][q]; M[r][q] = t; }
        const double t = b[c]; b[c] = b[r]; b[r] = t;
      }
    }
    const double ip = dp_rcp(M[c][c]);
#pragma unroll
    for (int r = c + 1; r < 4; ++r) {
      const double f = M[r][c] * ip;
#pragma unroll
      for (int q = c; q < 4; ++q) M[r][q] = fma(-f, M[c][q], M[r][q]);
      b[r] = fma(-f, b[c], b[r]);
    }
    M[c][c] = ip;                                            // keep the inverse pivot
  }
#pragma unroll
  for (int r = 3; r >= 0; --r) {
    double s = b[r];
#pragma unroll
    for (int q = r + 1; q < 4; ++q) s = fma(-M[r][q], b[q], s);
    b[r] = s * M[r][r];
  }
}

// per-lane constants of a mode
struct ModeK {
  double k, k2, kxt, kyt, sgI;       // |k|, (k H/2)^2, derivative multipliers (0 on the unpaired Nyquist index), sign of Re/Im(i z)
};

// ---- wall correction coefficients of a lane (own part), basis: 0 = z e^{-kz}, 1 = e^{-kz}, 2 = z e^{-k(H-z)}, 3 = e^{-k(H-z)}
//   wall data (eq 27 / (A3), u_wall uniform, i.e. absent for k != 0): u_0 = -u_DP(0) + l0 du_DP/dz(0), u_H = -u_DP(H) - lH du_DP/dz(H)
//   for the tangential components (slit; l0 = lH = 0 is no slip), w_0 = -w_DP(0), w_H = -w_DP(H); end values by direct summation:
//   y(0) = S_even - S_odd, y(H) = S_even + S_odd, (H/2) dy/dz likewise from the sums of the first-integral coefficients b_m
//   (even m come from the odd chain, odd m from the even chain; footnote 46).
//   Sums of this lane's columns: ssum[c * 2 + par] = S_c of (u, v, w)[c] from the even / odd chain, ssb[c * 2 + par] = S_b of (u, v)[c].
__device__ __forceinline__ void correction_coefficients(const double (&ssum)[6], const double (&ssb)[4], const ModeK& K,
                                                        double H, int wall_mode, double l0, double lH, double cf[3][4]) {
  double u0[3], uH[3], u0o[3], uHo[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double se = ssum[c * 2 + 0], so = ssum[c * 2 + 1];
    u0[c] = -(se - so); uH[c] = -(se + so);
  }
  if (wall_mode == DP_SLIT && (l0 != 0.0 || lH != 0.0)) {
    const double inv_s = 2.0 * dp_rcp(H);
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const double b_odd = ssb[c * 2 + 0], b_even = ssb[c * 2 + 1];   // from the even / odd chain
      u0[c] = fma(l0 * inv_s, b_even - b_odd, u0[c]);
      uH[c] = fma(-lH * inv_s, b_even + b_odd, uH[c]);
    }
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) { u0o[c] = __shfl_xor_sync(0xffffffffu, u0[c], 1); uHo[c] = __shfl_xor_sync(0xffffffffu, uH[c], 1); }
  const double k = K.k, kxt = K.kxt, kyt = K.kyt, sgI = K.sgI;
#pragma unroll
  for (int c = 0; c < 3; ++c) { cf[c][0] = cf[c][1] = cf[c][2] = cf[c][3] = 0.0; }
  if (wall_mode == DP_BOTTOM_WALL) {
    // eqs 42-44: Q = i k w0 + kx u0 + ky v0 ; Wc = k w0 - i kx u0 - i ky v0
    const double Q = fma(sgI * k, u0o[2], fma(kxt, u0[0], kyt * u0[1]));
    const double Wc = fma(k, u0[2], -sgI * fma(kxt, u0o[0], kyt * u0o[1]));
    const double ik = dp_rcp(k);
    cf[0][0] = -(kxt * ik) * Q; cf[1][0] = -(kyt * ik) * Q; cf[2][0] = Wc;
    cf[0][1] = u0[0]; cf[1][1] = u0[1]; cf[2][1] = u0[2];
  } else {
    // App. A.  Unknowns C0' = C0/(2 eta), D0' = D0 e^{kH}/(2 eta), C_c, D~_c = D_c e^{kH} (basis e^{-k(H-z)}, reading G13); e = e^{-kH}.
    // Tangential pairs, c = x, y ((A8a), (A8c)):
    //   a1 C_c + a2 D~_c = u0_c - i k_c (p1 C0' + p2 D0'),   a3 C_c + a4 D~_c = uH_c - i k_c (p3 C0' + p4 D0')
    //   a1 = 1 + k l0, a2 = (1 - k l0) e, a3 = (1 - k lH) e, a4 = 1 + k lH, p1 = l0/k, p2 = -l0 e/k,
    //   p3 = (H e/k)(k lH - lH/H - 1), p4 = (H/k)(k lH + lH/H + 1).
    // Eliminating them from the two continuity rows (A10a), (A10b) leaves a REAL 4x4 system for [C0', D0', Cz, D~z] with the rows
    // (A8b), (A8d), (A10a), (A10b); its right-hand sides are complex, one part per lane.
    const double e = dp_exp_neg(-k * H), ik = dp_rcp(k);
    const double a1 = 1.0 + k * l0, a2 = (1.0 - k * l0) * e, a3 = (1.0 - k * lH) * e, a4 = 1.0 + k * lH;
    const double p1 = l0 * ik, p2 = -l0 * e * ik, p3 = H * e * ik * (k * lH - lH * dp_rcp(H) - 1.0), p4 = H * ik * (k * lH + lH * dp_rcp(H) + 1.0);
    const double idet = dp_rcp(a1 * a4 - a2 * a3);
    const double g1a = (a4 - e * a3) * idet, g2a = (e * a1 - a2) * idet, g1b = (e * a4 - a3) * idet, g2b = (a1 - e * a2) * idet;
    const double kk = kxt * kxt + kyt * kyt;
    double M[4][4] = {{0.0, 0.0, 1.0, e},
                      {H * e, H, e, 1.0},
                      {1.0 + kk * (g1a * p1 + g2a * p3), e + kk * (g1a * p2 + g2a * p4), -k, k * e},
                      {e + kk * (g1b * p1 + g2b * p3), 1.0 + kk * (g1b * p2 + g2b * p4), -k * e, k}};
    // right-hand sides: [w0, wH, -i (g1a q0 + g2a qH), -i (g1b q0 + g2b qH)], q = kx u + ky v;  own part of -i z = -sgI * other part of z
    const double q0o = fma(kxt, u0o[0], kyt * u0o[1]), qHo = fma(kxt, uHo[0], kyt * uHo[1]);
    double b[4] = {u0[2], uH[2], -sgI * (g1a * q0o + g2a * qHo), -sgI * (g1b * q0o + g2b * qHo)};
    solve4(M, b);
    const double C0 = b[0], D0 = b[1];
    const double C0o = __shfl_xor_sync(0xffffffffu, C0, 1), D0o = __shfl_xor_sync(0xffffffffu, D0, 1);
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const double kc = c == 0 ? kxt : kyt;
      // own part of -i k_c X = -k_c sgI other(X)
      const double r1 = fma(-kc * sgI, p1 * C0o + p2 * D0o, u0[c]);
      const double r2 = fma(-kc * sgI, p3 * C0o + p4 * D0o, uH[c]);
      cf[c][1] = (a4 * r1 - a2 * r2) * idet;
      cf[c][3] = (a1 * r2 - a3 * r1) * idet;
      // (A5): -i (k_c/k) C0' z e^{-kz} + i (k_c/k) D0' z e^{-k(H-z)}
      cf[c][0] = -sgI * (kc * ik) * C0o;
      cf[c][2] = sgI * (kc * ik) * D0o;
    }
    // (A6): C0' z e^{-kz} + D0' z e^{-k(H-z)} + Cz e^{-kz} + Dz e^{-k(H-z)}
    cf[2][0] = C0; cf[2][2] = D0; cf[2][1] = b[2]; cf[2][3] = b[3];
  }
}

}  // namespace dp_solve
