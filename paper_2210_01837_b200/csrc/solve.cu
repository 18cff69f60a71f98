// solve.cu — per-wavenumber kernel of the doubly-periodic Stokes solver (paper steps 2(z)-6):
//   Chebyshev analysis in z (DCT-I), torque curl (eq 7), pressure BVP (eqs 15, 17), velocity BVPs (eqs 18, 22, 24),
//   wall correction (eqs 42-44 for one wall; App. A (A5),(A6),(A8),(A10) for the slit), (1/2) curl u (eq 11),
//   Chebyshev synthesis — all fused: every (kx,ky) column of every field is read from HBM once and written once.
//   The k = 0 column (eqs 47, 51, 52; (A12)) has its own small kernel.
//
// Discrete problem (identical to the oracle's): unknown polynomial of degree nz-1; tau rows 0..nz-3 of
// (D^2 - k^2) y = r plus the two Dirichlet-to-Neumann rows.  It is solved here in Greengard's integration form
// (ref [45]): unknowns a_n = Chebyshev coefficients of y'', first/second integrals b_n, c_n,
//   a_n - kappa^2 c_n = (H/2)^2 r_n,  kappa = k H/2,
// which couples a_{n-2}, a_n, a_{n+2} only ("pentadiagonal") = two diagonally dominant tridiagonal
// chains (n even / n odd), each with one border unknown (c_0 resp. b_0) fixed by one combination of the two
// boundary rows.  The chains are factored once per mode and reused for p, u, v, w.
//
// B200 mapping: one CTA = 16 consecutive modes of one row of the half spectrum, 6 warps.  A lane is (mode, part):
// lane = 2*mode + part, part 0 = real, 1 = imaginary, so a warp row of a complex column is 256 contiguous bytes in HBM
// and in shared memory ([column][n][lane], conflict free).  Every real operator of the method (cosine transforms,
// z-derivative, tridiagonal sweeps) acts on a lane's own 32 numbers only, so a warp that owns a column needs no
// synchronisation at all; the imaginary unit couples a lane to its neighbour (lane^1).  Work is split into phases of
// independent column items, one warp per item, sized so that 5-6 of the 6 warps are busy in every long phase; the
// sweeps run out of registers (all loads hoisted), divisions by constants are compile-time reciprocals, and the
// transform matrices are warp-uniform constant-bank operands of fully unrolled DFMAs (nz is a template parameter).
// Shared memory: 6 columns + 3 factor vectors = 61 KB at nz = 32 -> 3 CTAs (18 warps) per SM.
#include <cmath>
#include <vector>

#include "common.cuh"

namespace {

constexpr int TM = DP_SOLVE_TM;        // modes per CTA
constexpr int LN = 2 * TM;             // lanes of a complex column row (= 32)
constexpr int SOLVE_WARPS = 6;
constexpr int SOLVE_THREADS = SOLVE_WARPS * 32;
static_assert(LN == 32, "a warp row is one complex column row");

// ---- constant tables per compiled nz (N = nz-1, LH = nz/2):
//   CA[n][l] = cos(n l pi/N), l < LH                       analysis rows (contiguous in l)
//   SE[l][j] = cos(2j l pi/N), SO[l][j] = cos((2j+1) l pi/N), l, j < LH     synthesis rows (contiguous in j)
//   P[n], Q[n]: boundary-row functionals of a unit a_n (see chain()), XI[l] = cos(l pi/N)
template <int NZ> struct Tab {
  static constexpr int LH = NZ / 2;
  static constexpr int CA = 0, SE = CA + NZ * LH, SO = SE + LH * LH, P = SO + LH * LH, Q = P + NZ, XI = Q + NZ, SIZE = XI + NZ;
};
__constant__ double c_tab16[Tab<16>::SIZE];
__constant__ double c_tab32[Tab<32>::SIZE];
__constant__ double c_tab48[Tab<48>::SIZE];
template <int NZ> __device__ __forceinline__ const double* tab();
template <> __device__ __forceinline__ const double* tab<16>() { return c_tab16; }
template <> __device__ __forceinline__ const double* tab<32>() { return c_tab32; }
template <> __device__ __forceinline__ const double* tab<48>() { return c_tab48; }

struct SolveArgs {
  double2* cplx;
  size_t cplx_field;
  int nx, ny, nkx;
  int n_fast, n_slow, pitch;     // half spectrum stored as [field][l][slow][fast (pitch)]
  int fast_is_x;                 // 1: fast index = kx index (cuFFT layout); 0: fast index = position along ky (transposed layout)
  const int* lmin;               // planes l < *lmin of the input hold zeros that were never written: not read
  const int* ky_of_pos;          // transposed layout: FFT-order ky index stored at each position (digit reversal of the y pass), or null
  double Lx, Ly, H, eta;
  int wall_mode, torque, omega;
};

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---- tridiagonal rows of a chain (n >= 1): d_n a_n + l_n a_{n-2} + u_n a_{n+2}; all divisions are compile-time constants
template <int NZ> __device__ __forceinline__ double row_d(int n, double k2) { return n == 1 ? fma(k2, 0.125, 1.0) : fma(k2, 1.0 / (2.0 * (n * n - 1)), 1.0); }
template <int NZ> __device__ __forceinline__ double row_l(int n, double k2) { return k2 * (-(n == 2 ? 2.0 : 1.0) / (4.0 * n * (n - 1))); }
template <int NZ> __device__ __forceinline__ double row_u(int n, double k2) { return (n + 2 <= NZ - 3) ? k2 * (-1.0 / (4.0 * n * (n + 1))) : 0.0; }

// ---- DCT-I analysis of a lane's column, in place:
//   g^_n = (2/N)(1/c~_n) sum_l (1/c~_l) g_l cos(n l pi/N), folded with cos(n (N-l) pi/N) = (-1)^n cos(n l pi/N)
template <int NZ> __device__ __forceinline__ void analysis_column(double* __restrict__ v) {
  constexpr int N = NZ - 1, LH = NZ / 2;
  const double* __restrict__ T = tab<NZ>() + Tab<NZ>::CA;
  double e[LH], o[LH];
#pragma unroll
  for (int l = 0; l < LH; ++l) {
    const double a = v[l * LN], b = v[(N - l) * LN];
    e[l] = a + b; o[l] = a - b;
  }
  e[0] *= 0.5; o[0] *= 0.5;
#pragma unroll
  for (int j = 0; j < LH; ++j) {
    double ae0 = 0.0, ae1 = 0.0, ao0 = 0.0, ao1 = 0.0;      // two partial sums per output (see synthesis_column)
#pragma unroll
    for (int l = 0; l < LH; l += 2) {
      ae0 = fma(T[(2 * j) * LH + l], e[l], ae0); ae1 = fma(T[(2 * j) * LH + l + 1], e[l + 1], ae1);
      ao0 = fma(T[(2 * j + 1) * LH + l], o[l], ao0); ao1 = fma(T[(2 * j + 1) * LH + l + 1], o[l + 1], ao1);
    }
    const double ae = ae0 + ae1, ao = ao0 + ao1;
    v[(2 * j) * LN] = ae * (j == 0 ? 1.0 / N : 2.0 / N);
    v[(2 * j + 1) * LN] = ao * ((2 * j + 1 == N) ? 1.0 / N : 2.0 / N);
  }
}

// ---- DCT-I synthesis of a lane's column, in place: g_l = sum_n g^_n cos(n l pi/N)
template <int NZ> __device__ __forceinline__ void synthesis_column(double* __restrict__ v) {
  constexpr int N = NZ - 1, LH = NZ / 2;
  const double* __restrict__ TE = tab<NZ>() + Tab<NZ>::SE;
  const double* __restrict__ TO = tab<NZ>() + Tab<NZ>::SO;
  double ce[LH], co[LH];
#pragma unroll
  for (int j = 0; j < LH; ++j) { ce[j] = v[(2 * j) * LN]; co[j] = v[(2 * j + 1) * LN]; }
  // two partial sums per output: with a single dependent chain per output the compiler interleaves many outputs and then
  // spends one uniform-register move per DFMA on juggling the table operands
#pragma unroll
  for (int l = 0; l < LH; ++l) {
    double E0 = 0.0, E1 = 0.0, O0 = 0.0, O1 = 0.0;
#pragma unroll
    for (int j = 0; j < LH; j += 2) {
      E0 = fma(TE[l * LH + j], ce[j], E0); E1 = fma(TE[l * LH + j + 1], ce[j + 1], E1);
      O0 = fma(TO[l * LH + j], co[j], O0); O1 = fma(TO[l * LH + j + 1], co[j + 1], O1);
    }
    const double E = E0 + E1, O = O0 + O1;
    v[l * LN] = E + O;
    v[(N - l) * LN] = E - O;
  }
}

// ---- coefficient-space z-derivative of a lane's column (both parities), top-down recurrence
//   d_N = 0, d_n = d_{n+2} + 2(n+1) g_{n+1},  (D g)_n = (2/H) d_n (d_0 halved);  dst[n] (+)= scale * (D src)_n
template <int NZ, bool ACC> __device__ __forceinline__ void deriv_column(const double* __restrict__ src, double* __restrict__ dst, double inv_s, double scale) {
  constexpr int N = NZ - 1;
  double g[NZ];
#pragma unroll
  for (int n = 1; n <= N; ++n) g[n] = src[n * LN];
  double d0 = 0.0, d1 = 0.0;          // running sums of the two parities
  const double f = inv_s * scale;
#pragma unroll
  for (int n = N; n >= 0; --n) {
    double& d = (n & 1) ? d1 : d0;
    if (n + 1 <= N) d = fma(2.0 * (n + 1), g[n + 1], d);
    const double val = d * (n == 0 ? 0.5 * f : f);
    if (ACC) dst[n * LN] += val; else dst[n * LN] = val;
  }
}

// ---- chain geometry: rows n0, n0+2, ... <= N-2 of parity PAR
template <int NZ, int PAR> struct Ch {
  static constexpr int N = NZ - 1, n0 = PAR ? 1 : 2, NR = PAR ? (N - 1) / 2 : (N - 2) / 2;
};

// ---- factorisation of one chain and its homogeneous ("border") solution, per mode (depends on |k| only):
//   Fm[n] = Thomas multiplier, Fi[n] = inverse pivot, Fa[n] = a_n of the solution with unit border unknown,
//   returns 1/B_g, B_g = boundary functional of that solution.
template <int NZ, int PAR>
__device__ __forceinline__ double factor_chain(double* __restrict__ Fm, double* __restrict__ Fi, double* __restrict__ Fa, double k, double k2,
                                               double inv_s, bool store) {
  constexpr int n0 = Ch<NZ, PAR>::n0, NR = Ch<NZ, PAR>::NR;
  const double* __restrict__ T = tab<NZ>();
  double invd[NR], ag[NR];
  double g = PAR ? k2 : 0.25 * k2 * k2;
#pragma unroll
  for (int j = 0; j < NR; ++j) {
    const int n = n0 + 2 * j;
    double d = row_d<NZ>(n, k2);
    if (j > 0) {
      const double mu = row_l<NZ>(n, k2) * invd[j - 1];
      d = fma(-mu, row_u<NZ>(n - 2, k2), d);
      if (store) Fm[n * TM] = mu;
      g = -mu * g;
    }
    invd[j] = 1.0 / d;
    ag[j] = g;
  }
  double SP = 0.0, SQ = 0.0, next = 0.0;
#pragma unroll
  for (int j = NR - 1; j >= 0; --j) {
    const int n = n0 + 2 * j;
    const double a = (ag[j] - row_u<NZ>(n, k2) * next) * invd[j];
    next = a;
    if (store) { Fa[n * TM] = a; Fi[n * TM] = invd[j]; }
    SP = fma(T[Tab<NZ>::P + n], a, SP); SQ = fma(T[Tab<NZ>::Q + n], a, SQ);
  }
  double Bg;
  if (!PAR) {                                                // a_0 = rho_0 + kappa^2 c_0 ; c_0 = 1 also enters sum c_n directly
    SP = fma(T[Tab<NZ>::P + 0], k2, SP); SQ = fma(T[Tab<NZ>::Q + 0], k2, SQ);
    Bg = inv_s * SP + k * (1.0 + SQ);
  } else {                                                   // b_0 = 1 enters sum b_n and c_1
    Bg = inv_s * (1.0 + SP) + k * (1.0 + SQ);
  }
  return 1.0 / Bg;
}

// ---- one chain of one BVP for a lane: forward elimination, back substitution with the boundary functional, border
//      unknown, double integration.  a[j] = (H/2)^2 r_n of row n = n0+2j on entry, rho0 = (H/2)^2 r_0 (even chain).
//      Writes y's coefficients c_n of parity PAR to col and, if WITH_D, the coefficients of dy/dz of the OTHER parity to
//      dcol.  Returns S_c = sum of the c_n written (incl. c_0 for the even chain).
template <int NZ, int PAR>
__device__ __forceinline__ double chain(bool WITH_D, double (&a)[Ch<NZ, PAR>::NR], double rho0, const double* __restrict__ Fm, const double* __restrict__ Fi,
                                        const double* __restrict__ Fa, double* __restrict__ col, double* __restrict__ dcol, double k,
                                        double k2, double inv_s, double beta_bc, double invBg) {
  constexpr int N = NZ - 1, n0 = Ch<NZ, PAR>::n0, NR = Ch<NZ, PAR>::NR;
  const double* __restrict__ T = tab<NZ>();
  double mult[NR], invd[NR], ag[NR];
#pragma unroll
  for (int j = 0; j < NR; ++j) {
    const int n = n0 + 2 * j;
    mult[j] = j > 0 ? Fm[n * TM] : 0.0; invd[j] = Fi[n * TM]; ag[j] = Fa[n * TM];
  }
  if (!PAR) a[0] = fma(0.25 * k2, rho0, a[0]);               // even chain: row 2 carries (kappa^2/4) rho_0
#pragma unroll
  for (int j = 1; j < NR; ++j) a[j] = fma(-mult[j], a[j - 1], a[j]);
  double SP = 0.0, SQ = 0.0, next = 0.0;
#pragma unroll
  for (int j = NR - 1; j >= 0; --j) {
    const int n = n0 + 2 * j;
    const double v = (a[j] - row_u<NZ>(n, k2) * next) * invd[j];
    a[j] = v; next = v;
    SP = fma(T[Tab<NZ>::P + n], v, SP); SQ = fma(T[Tab<NZ>::Q + n], v, SQ);
  }
  if (!PAR) { SP = fma(T[Tab<NZ>::P + 0], rho0, SP); SQ = fma(T[Tab<NZ>::Q + 0], rho0, SQ); }
  const double border = (beta_bc - (inv_s * SP + k * SQ)) * invBg;       // c_0 (even chain) or b_0 (odd chain)
#pragma unroll
  for (int j = 0; j < NR; ++j) a[j] = fma(border, ag[j], a[j]);
  // integrate twice:  b_{n+1} = (cbar_n a_n - a_{n+2}) / (2(n+1)),  c_n = (cbar_{n-1} b_{n-1} - b_{n+1}) / (2n)
  double Sc = 0.0, bprev;
  if (!PAR) { col[0] = border; Sc = border; bprev = 0.0; }
  else { bprev = border; if (WITH_D) dcol[0] = border * inv_s; }
#pragma unroll
  for (int i = 0; i <= (N - PAR) / 2; ++i) {
    const int n = PAR + 2 * i;
    // a_n of parity PAR: n = 0 -> rho0 + border kappa^2 (even); n = n0 + 2j -> a[j]; n > N-2 -> 0
    double an = 0.0, ap = 0.0;
    if (n <= N - 2) an = (!PAR && n == 0) ? fma(border, k2, rho0) : a[n >= n0 ? (n - n0) / 2 : 0];
    if (n + 2 <= N - 2) ap = a[(n + 2 - n0) / 2];
    const double bn1 = ((n == 0 ? 2.0 : 1.0) * an - ap) * (1.0 / (2.0 * (n + 1)));
    if (n >= 1) {
      const double c = ((n == 1 ? 2.0 : 1.0) * bprev - bn1) * (1.0 / (2.0 * n));
      col[n * LN] = c;
      Sc += c;
    }
    if (WITH_D && n + 1 <= N - 1) dcol[(n + 1) * LN] = bn1 * inv_s;
    bprev = bn1;
  }
  if (WITH_D && ((N - PAR) & 1) == 1) dcol[N * LN] = 0.0;    // (D y)_N = 0: slot N belongs to the chain whose b's have N's parity
  return Sc;
}

// ---- 4x4 real system, one right-hand side per lane, partial pivoting after row equilibration
__device__ __forceinline__ void solve4(double M[4][4], double b[4]) {
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    const double mx = fmax(fmax(fabs(M[r][0]), fabs(M[r][1])), fmax(fabs(M[r][2]), fabs(M[r][3])));
    const double s = mx > 0.0 ? 1.0 / mx : 1.0;
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
    const double ip = 1.0 / M[c][c];
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

// ---- one BVP item of a lane: kind 0 = pressure (eqs 15, 17): right-hand side i k.f + dz f_z, p -> C3, dp/dz -> C4;
//      kind 1 = u or v (comp 0, 1), kind 2 = w (eq 18 with BCs 22, 24): f_c (column comp) is overwritten by u_c.
//      One code path per parity so that the chain sweeps exist once in the instruction stream.
template <int NZ, int PAR>
__device__ __noinline__ double bvp_item(int kind, int comp, double* __restrict__ C, const double* __restrict__ F, int lane, int mode, ModeK K,
                                        double s, double inv_s, double eta, double invBg, double pH_own, double p0_own, double pH_oth, double p0_oth) {
  constexpr int N = NZ - 1, n0 = Ch<NZ, PAR>::n0, NR = Ch<NZ, PAR>::NR, VS = NZ * LN;
  double a[NR], rho0 = 0.0, beta_bc = 0.0;
  double* col;
  if (kind == 0) {
    const double* fxo = C + 0 * VS + (lane ^ 1);          // the OTHER part of f_x, f_y: i k f mixes re and im
    const double* fyo = C + 1 * VS + (lane ^ 1);
    const double* fz = C + 2 * VS + lane;
    double d = 0.0;
    constexpr int ntop = ((N - PAR) & 1) ? N - 1 : N;     // largest n <= N with parity PAR
    const double s2 = s * s;
#pragma unroll
    for (int i = 0; i <= ntop / 2; ++i) {
      const int n = ntop - 2 * i;
      if (n < 0) break;
      if (n + 1 <= N) d = fma(2.0 * (n + 1), fz[(n + 1) * LN], d);
      if (n <= N - 2) {
        const double r = fma(K.sgI, fma(K.kxt, fxo[n * LN], K.kyt * fyo[n * LN]), d * (n == 0 ? 0.5 * inv_s : inv_s)) * s2;
        if (n >= n0) a[n >= n0 ? (n - n0) / 2 : 0] = r; else rho0 = r;
      }
    }
    col = C + 3 * VS + lane;
  } else {
    col = C + comp * VS + lane;
    const double sc = s * s / eta;
    double gH, g0;
    // kind 1: r = (i k_c p - f_c)/eta ; kind 2: r = (dz p - f_z)/eta
    const double* src = kind == 1 ? C + 3 * VS + (lane ^ 1) : C + 4 * VS + lane;
    const double kc = comp == 0 ? K.kxt : K.kyt;
    const double f = kind == 1 ? K.sgI * kc : 1.0;
#pragma unroll
    for (int i = 0; i <= (N - 2 - PAR) / 2; ++i) {
      const int n = PAR + 2 * i;
      const double r = (f * src[n * LN] - col[n * LN]) * sc;
      if (n >= n0) a[n >= n0 ? (n - n0) / 2 : 0] = r; else rho0 = r;
    }
    if (kind == 1) {
      // (dz + k) u(H) = -(i k_c/(2 k eta)) p(H) ; (dz - k) u(0) = +(i k_c/(2 k eta)) p(0)      (eq 22)
      const double c = kc / (2.0 * K.k * eta);
      gH = -K.sgI * c * pH_oth; g0 = K.sgI * c * p0_oth;
    } else {
      // (dz + k) w(H) = p(H)/(2 eta) ; (dz - k) w(0) = p(0)/(2 eta)                              (eq 24)
      gH = pH_own / (2.0 * eta); g0 = p0_own / (2.0 * eta);
    }
    beta_bc = PAR ? 0.5 * (gH + g0) : 0.5 * (gH - g0);
  }
  return chain<NZ, PAR>(kind == 0, a, rho0, F + 0 * NZ * TM + mode, F + 1 * NZ * TM + mode, F + 2 * NZ * TM + mode, col, C + 4 * VS + lane,
                        K.k, K.k2, inv_s, beta_bc, invBg);
}

// ---- wall correction coefficients of a lane (own part), basis: 0 = z e^{-kz}, 1 = e^{-kz}, 2 = z e^{-k(H-z)}, 3 = e^{-k(H-z)}
//   wall data (eq 27 / (A3) with no slip, u_wall = 0): u_0 = -u_DP(z=0) = -(S_even - S_odd), u_H = -u_DP(z=H) = -(S_even + S_odd)
__device__ __forceinline__ void correction_coefficients(const double* __restrict__ s_sum, int lane, const ModeK& K, double H, int wall_mode,
                                                        double cf[3][4]) {
  double u0[3], uH[3], u0o[3], uHo[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double se = s_sum[((1 + c) * 2 + 0) * LN + lane], so = s_sum[((1 + c) * 2 + 1) * LN + lane];
    u0[c] = -(se - so); uH[c] = -(se + so);
    u0o[c] = __shfl_xor_sync(0xffffffffu, u0[c], 1); uHo[c] = __shfl_xor_sync(0xffffffffu, uH[c], 1);
  }
  const double k = K.k, kxt = K.kxt, kyt = K.kyt, sgI = K.sgI;
#pragma unroll
  for (int c = 0; c < 3; ++c) { cf[c][0] = cf[c][1] = cf[c][2] = cf[c][3] = 0.0; }
  if (wall_mode == DP_BOTTOM_WALL) {
    // eqs 42-44: Q = i k w0 + kx u0 + ky v0 ; Wc = k w0 - i kx u0 - i ky v0
    const double Q = fma(sgI * k, u0o[2], fma(kxt, u0[0], kyt * u0[1]));
    const double Wc = fma(k, u0[2], -sgI * fma(kxt, u0o[0], kyt * u0o[1]));
    const double ik = 1.0 / k;
    cf[0][0] = -(kxt * ik) * Q; cf[1][0] = -(kyt * ik) * Q; cf[2][0] = Wc;
    cf[0][1] = u0[0]; cf[1][1] = u0[1]; cf[2][1] = u0[2];
  } else {
    // App. A, no slip.  Unknowns [C0', D0', Cz, Dz] with C0' = C0/(2 eta), D0' = D0 e^{kH}/(2 eta) (basis e^{-k(H-z)}):
    // (A8b), (A8d), (A10a), (A10b) after eliminating Cx+e Dx, e Cx+Dx (and y) with (A8a), (A8c); e = e^{-kH}.
    const double e = exp(-k * H), ik = 1.0 / k;
    const double g = (kxt * kxt + kyt * kyt) * H * ik;
    double M[4][4] = {{0.0, 0.0, 1.0, e}, {H * e, H, e, 1.0}, {1.0, e, -k, k * e}, {e * (1.0 - g), 1.0 + g, -k * e, k}};
    // right-hand sides: [w0, wH, -i(kx u0 + ky v0), -i(kx uH + ky vH)]  ->  own part of -i z = -sgI * other part of z
    double b[4] = {u0[2], uH[2], -sgI * fma(kxt, u0o[0], kyt * u0o[1]), -sgI * fma(kxt, uHo[0], kyt * uHo[1])};
    solve4(M, b);
    const double C0 = b[0], D0 = b[1];
    const double C0o = __shfl_xor_sync(0xffffffffu, C0, 1), D0o = __shfl_xor_sync(0xffffffffu, D0, 1);
    const double iom = 1.0 / (-expm1(-k * H) * (1.0 + e));       // 1/(1 - e^2)
#pragma unroll
    for (int c = 0; c < 2; ++c) {
      const double kc = c == 0 ? kxt : kyt, q = kc * H * ik;
      // C_c + e D_c = u0 ; e C_c + D_c = uH + i q (e C0' - D0')
      const double r2 = fma(sgI * q, e * C0o - D0o, uH[c]);
      cf[c][1] = (u0[c] - e * r2) * iom;
      cf[c][3] = (r2 - e * u0[c]) * iom;
      // (A5): -i (k_c/k) C0' z e^{-kz} + i (k_c/k) D0' z e^{-k(H-z)}
      cf[c][0] = -sgI * (kc * ik) * C0o;
      cf[c][2] = sgI * (kc * ik) * D0o;
    }
    // (A6): C0' z e^{-kz} + D0' z e^{-k(H-z)} + Cz e^{-kz} + Dz e^{-k(H-z)}
    cf[2][0] = C0; cf[2][2] = D0; cf[2][1] = b[2]; cf[2][3] = b[3];
  }
}

template <int NZ> struct SolveSmem {
  static constexpr int VS = NZ * LN;                                   // one complex column [n][lane]
  static constexpr int COLS = 6 * VS;                                  // C0..C5
  static constexpr int FACT = COLS;                                    // [3][NZ][TM]: multipliers, inverse pivots, border solution
  static constexpr int IBG = FACT + 3 * NZ * TM;                       // [2][TM] 1/B_g of the even / odd chain
  static constexpr int SUM = IBG + 2 * TM;                             // [4][2][LN] S_c of (p,u,v,w) x (even, odd chain)
  static constexpr int CORR = SUM + 8 * LN;                            // [12][LN] correction coefficients (slit)
  static constexpr int DOUBLES = CORR + 12 * LN;
};

#ifdef DP_SOLVE_TIMING
// phase timeline of the CTAs that run on a few SMs (development builds only)
__device__ long long g_tlog[4 * 256 * SOLVE_WARPS * 16];
__device__ int g_tcount[4];
#define TMARK(k) do { if (tslot >= 0 && lane == 0) g_tlog[((tsm * 256 + tslot) * SOLVE_WARPS + wid) * 16 + (k)] = clock64(); } while (0)
#else
#define TMARK(k) do { } while (0)
#endif

template <int NZ>
__global__ void __launch_bounds__(SOLVE_THREADS, (NZ <= 32 ? 3 : 2)) k_solve(SolveArgs A) {
  extern __shared__ double smem[];
  constexpr int N = NZ - 1, VS = NZ * LN;
  typedef SolveSmem<NZ> S;
  double* C = smem;                      // columns: 0 f_x->u, 1 f_y->v, 2 f_z->w, 3 t_x->p->dz u, 4 t_y->dz p->dz v, 5 (E, zE)
  double* F = smem + S::FACT;
  double* s_ibg = smem + S::IBG;
  double* s_sum = smem + S::SUM;
  double* s_corr = smem + S::CORR;
  const double* T = tab<NZ>();

  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int mode = lane >> 1, part = lane & 1;
#ifdef DP_SOLVE_TIMING
  __shared__ int s_tslot;
  int tsm = -1, tslot = -1;
  {
    unsigned smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    if (smid < 4) {
      tsm = (int)smid;
      if (tid == 0) { const int c = atomicAdd(&g_tcount[smid], 1); s_tslot = c < 256 ? c : -1; }
      __syncthreads();
      tslot = s_tslot;
    }
  }
  TMARK(0);
#endif
  const int ifast = blockIdx.x * TM + mode, islow = blockIdx.y;
  const bool valid = ifast < A.n_fast;
  const int ix = A.fast_is_x ? ifast : islow;
  const int iy = A.fast_is_x ? islow : ((A.ky_of_pos && valid) ? __ldg(A.ky_of_pos + ifast) : ifast);
  const bool zero_mode = (ix == 0 && iy == 0);
  const double s = 0.5 * A.H, inv_s = 1.0 / s, eta = A.eta;
  ModeK K;
  K.k = 1.0; K.kxt = 0.0; K.kyt = 0.0; K.sgI = part ? 1.0 : -1.0;
  if (valid && !zero_mode) {
    const int nyq = (iy <= A.ny / 2) ? iy : iy - A.ny;
    const double kx = 2.0 * M_PI * ix / A.Lx, ky = 2.0 * M_PI * nyq / A.Ly;
    K.k = sqrt(kx * kx + ky * ky);                         // magnitude: always the full values (reading G5)
    K.kxt = (ix == A.nx / 2) ? 0.0 : kx;                   // component multipliers vanish on the unpaired Nyquist index
    K.kyt = (iy == A.ny / 2) ? 0.0 : ky;
  }
  K.k2 = (K.k * s) * (K.k * s);
  const size_t plane = (size_t)A.n_slow * A.pitch;
  const size_t off0 = (size_t)islow * A.pitch + ifast;
  const double* gin = reinterpret_cast<const double*>(A.cplx);

  // ---------------- phase 0: all nodal columns go HBM -> shared memory as 8-byte cp.async (no registers, everything in
  // flight at once); t_z is only needed for the fold and travels through registers.  While the loads fly: warps 0, 1 factor
  // the two chains, warps 2-5 evaluate e^{-k z_l} and z_l e^{-k z_l} at the nodes (-> C5).  Then every warp folds the
  // algebraic part of (1/2) curl t into f for the rows it loaded itself (eq 7).
  constexpr int ROWS = (NZ + SOLVE_WARPS - 1) / SOLVE_WARPS;
  const int lm = __ldg(A.lmin);
  double tz[ROWS];
#pragma unroll
  for (int r = 0; r < ROWS; ++r) {
    const int l = wid + r * SOLVE_WARPS;
    tz[r] = 0.0;
    if (l < NZ) {
      const int o = l * LN + lane;
      if (valid && l >= lm) {
        const size_t og = 2 * (l * plane + off0) + part;
#pragma unroll
        for (int c = 0; c < 3; ++c) cp_async8(&C[c * VS + o], &gin[2 * (c * A.cplx_field) + og]);
        if (A.torque) {
          cp_async8(&C[3 * VS + o], &gin[2 * (3 * A.cplx_field) + og]);
          cp_async8(&C[4 * VS + o], &gin[2 * (4 * A.cplx_field) + og]);
          tz[r] = __ldg(&gin[2 * (5 * A.cplx_field) + og]);
        }
      } else {
#pragma unroll
        for (int c = 0; c < 5; ++c) C[c * VS + o] = 0.0;
      }
    }
  }
  cp_async_commit();
  TMARK(1);
  if (wid == 0) {
    const double ib = factor_chain<NZ, 0>(F + mode, F + NZ * TM + mode, F + 2 * NZ * TM + mode, K.k, K.k2, inv_s, part == 0);
    if (part == 0) s_ibg[mode] = ib;
  } else if (wid == 1) {
    const double ib = factor_chain<NZ, 1>(F + mode, F + NZ * TM + mode, F + 2 * NZ * TM + mode, K.k, K.k2, inv_s, part == 0);
    if (part == 0) s_ibg[TM + mode] = ib;
  } else {
    for (int l = wid - 2; l < NZ; l += SOLVE_WARPS - 2) {
      const double zl = s * (1.0 + T[Tab<NZ>::XI + l]);
      const double E = exp(-K.k * zl);
      C[5 * VS + l * LN + lane] = part ? zl * E : E;
    }
  }
  TMARK(2);
  cp_async_wait_all();
  __syncwarp();
  if (A.torque) {
#pragma unroll
    for (int r = 0; r < ROWS; ++r) {
      const int l = wid + r * SOLVE_WARPS;
      if (l < NZ) {
        const int o = l * LN + lane, oo = l * LN + (lane ^ 1);
        const double t2o = __shfl_xor_sync(0xffffffffu, tz[r], 1);
        const double t0o = C[3 * VS + oo], t1o = C[4 * VS + oo];
        C[0 * VS + o] = fma(0.5 * K.sgI * K.kyt, t2o, C[0 * VS + o]);                       // f_x += (1/2) i k_y t_z
        C[1 * VS + o] = fma(-0.5 * K.sgI * K.kxt, t2o, C[1 * VS + o]);                      // f_y -= (1/2) i k_x t_z
        C[2 * VS + o] = fma(0.5 * K.sgI, K.kxt * t1o - K.kyt * t0o, C[2 * VS + o]);         // f_z += (1/2) i (k_x t_y - k_y t_x)
      }
    }
  }
  TMARK(3);
  __syncthreads();

  // ---------------- phase 1: Chebyshev analysis, one warp per column: f_x, f_y, f_z, (E, zE) [, t_x, t_y]   (step 2; step 6)
  {
    const int col = wid < 3 ? wid : (wid == 3 ? 5 : wid - 1);          // warps 0-2: C0-C2, warp 3: C5, warps 4, 5: C3, C4
    if (wid < 4 || A.torque) analysis_column<NZ>(C + col * VS + lane);
  }
  TMARK(4);
  __syncthreads();

  // ---------------- phase 2: f_x -= (1/2) D t_y, f_y += (1/2) D t_x (eq 7)
  if (A.torque) {
    if (wid < 2) deriv_column<NZ, true>(C + (wid == 0 ? 4 : 3) * VS + lane, C + wid * VS + lane, inv_s, wid == 0 ? -0.5 : 0.5);
    TMARK(5);
    __syncthreads();
  }

  // ---------------- phases 3, 4: pressure BVP (eqs 15, 17), one warp per chain; then the velocity BVPs (eq 18) with BCs
  // (22), (24), one warp per (component, chain)
#pragma unroll 1
  for (int ph = 0; ph < 2; ++ph) {
    if (ph == 1 || wid < 2) {
      const int comp = wid >> 1, par = wid & 1;
      const int kind = ph == 0 ? 0 : (comp == 2 ? 2 : 1);
      double pH = 0.0, p0 = 0.0;
      if (ph == 1) {
        const double se = s_sum[0 * LN + lane], so = s_sum[1 * LN + lane];
        pH = se + so; p0 = se - so;                       // p(H) = sum p_n, p(0) = sum (-1)^n p_n  ("direct summation")
      }
      const double pHo = __shfl_xor_sync(0xffffffffu, pH, 1), p0o = __shfl_xor_sync(0xffffffffu, p0, 1);
      double Sc;
      if (par) Sc = bvp_item<NZ, 1>(kind, comp, C, F, lane, mode, K, s, inv_s, eta, s_ibg[TM + mode], pH, p0, pHo, p0o);
      else Sc = bvp_item<NZ, 0>(kind, comp, C, F, lane, mode, K, s, inv_s, eta, s_ibg[mode], pH, p0, pHo, p0o);
      s_sum[((ph == 0 ? 0 : 1 + comp) * 2 + par) * LN + lane] = Sc;
    }
    TMARK(6 + ph);
    __syncthreads();
  }

  // ---------------- phase 5: correction coefficients (bottom wall: every warp for itself; slit: warp 0, shared)
  double cf[3][4];
  if (A.wall_mode == DP_BOTTOM_WALL) {
    correction_coefficients(s_sum, lane, K, A.H, DP_BOTTOM_WALL, cf);
  } else {
    if (wid == 0) {
      correction_coefficients(s_sum, lane, K, A.H, DP_SLIT, cf);
#pragma unroll
      for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 4; ++b) s_corr[(c * 4 + b) * LN + lane] = cf[c][b];
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int b = 0; b < 4; ++b) cf[c][b] = s_corr[(c * 4 + b) * LN + lane];
  }

  // ---------------- phase 6: total coefficients = DP + correction;  T[z e^{-k(H-z)}]_n = (-1)^n (H e_n - ze_n), T[e^{-k(H-z)}]_n = (-1)^n e_n
  for (int n = wid; n < NZ; n += SOLVE_WARPS) {
    const double mine = C[5 * VS + n * LN + lane], other = C[5 * VS + n * LN + (lane ^ 1)];
    const double en = part ? other : mine, zen = part ? mine : other;
    const double sgn = (n & 1) ? -1.0 : 1.0;
    const double b2 = sgn * (A.H * en - zen), b3 = sgn * en;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double add = fma(cf[c][0], zen, cf[c][1] * en);
      if (A.wall_mode == DP_SLIT) add = fma(cf[c][2], b2, fma(cf[c][3], b3, add));
      C[c * VS + n * LN + lane] += add;
    }
  }
  TMARK(8);
  __syncthreads();

  // ---------------- phase 7: dz u, dz v of the TOTAL in coefficient space (reading G12) -> C3, C4; synthesis back to the nodes
  if (A.omega) {
    if (wid < 2) deriv_column<NZ, false>(C + wid * VS + lane, C + (3 + wid) * VS + lane, inv_s, 1.0);
    TMARK(9);
    __syncthreads();
  }
  if (wid < (A.omega ? 5 : 3)) synthesis_column<NZ>(C + wid * VS + lane);
  TMARK(10);
  __syncthreads();

  // ---------------- phase 8: (1/2) curl u (eq 11), scale by 1/(nx ny) for the unnormalised inverse FFT, store
  const double scl = 1.0 / ((double)A.nx * (double)A.ny);
  double* gout = reinterpret_cast<double*>(A.cplx);
  for (int l = wid; l < NZ; l += SOLVE_WARPS) {
    const int o = l * LN + lane;
    const double u = C[0 * VS + o], v = C[1 * VS + o], w = C[2 * VS + o];
    double om[3] = {0, 0, 0};
    if (A.omega) {
      const double du = C[3 * VS + o], dv = C[4 * VS + o];
      const double uo = __shfl_xor_sync(0xffffffffu, u, 1), vo = __shfl_xor_sync(0xffffffffu, v, 1), wo = __shfl_xor_sync(0xffffffffu, w, 1);
      om[0] = 0.5 * (K.sgI * K.kyt * wo - dv);                          // (1/2)(i k_y w - dz v)
      om[1] = 0.5 * (du - K.sgI * K.kxt * wo);                          // (1/2)(dz u - i k_x w)
      om[2] = 0.5 * K.sgI * (K.kxt * vo - K.kyt * uo);                  // (1/2)(i k_x v - i k_y u)
    }
    if (valid && !zero_mode) {
      const size_t og = 2 * (l * plane + off0) + part;
      gout[2 * (0 * A.cplx_field) + og] = u * scl;
      gout[2 * (1 * A.cplx_field) + og] = v * scl;
      gout[2 * (2 * A.cplx_field) + og] = w * scl;
      if (A.omega) {
#pragma unroll
        for (int c = 0; c < 3; ++c) gout[2 * ((3 + c) * A.cplx_field) + og] = om[c] * scl;
      }
    }
  }
  TMARK(11);
}

#ifdef DP_SOLVE_TIMING
}  // namespace
extern "C" int dp_debug_solve_timeline(long long* host_log, int* host_count) {   // development builds only
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(host_log, g_tlog, sizeof(g_tlog));
  cudaMemcpyFromSymbol(host_count, g_tcount, sizeof(g_tcount));
  int z[4] = {0, 0, 0, 0};
  cudaMemcpyToSymbol(g_tcount, z, sizeof(z));
  return 0;
}
namespace {
#endif

// ---- k = 0 column (paper step 5; eqs 47, 51, 52; (A12) with no slip): one CTA of 64 threads
//   w = 0;  u'' = -f_x/eta, v'' = -f_y/eta with u(0) = 0 and (bottom wall) u'(H) = 0 / (slit) u(H) = 0.
//   With torques the k = 0 force is f_x - (1/2) dz t_y, f_y + (1/2) dz t_x (eq 7).
__global__ void k_zero_mode(SolveArgs A, int nz, const double* __restrict__ ct_full /* cos(n l pi/N) [nz][nz] */) {
  __shared__ double fc[4][2][DP_MAX_NZ];     // coefficients: f_x, f_y, t_x, t_y (re, im)
  __shared__ double uc[2][2][DP_MAX_NZ];     // u, v coefficients
  __shared__ double ub[2][2][DP_MAX_NZ];     // first-integral coefficients b_n (= (H/2) * du/dz coefficients)
  const int N = nz - 1, t = threadIdx.x;
  const double s = 0.5 * A.H;
  // analysis by direct summation
  for (int idx = t; idx < 4 * nz; idx += blockDim.x) {
    const int q = idx / nz, n = idx % nz;
    const int field = q < 2 ? q : (q == 2 ? 3 : 4);
    double ar = 0.0, ai = 0.0;
    if (q < 2 || A.torque) {
      for (int l = A.lmin[0] < 0 ? 0 : A.lmin[0]; l < nz; ++l) {
        double2 v = A.cplx[field * A.cplx_field + (size_t)l * A.n_slow * A.pitch];
        double wgt = ct_full[n * nz + l] * ((l == 0 || l == N) ? 0.5 : 1.0);
        ar += wgt * v.x; ai += wgt * v.y;
      }
      double sc = ((n == 0 || n == N) ? 1.0 : 2.0) / N;
      ar *= sc; ai *= sc;
    }
    fc[q][0][n] = ar; fc[q][1][n] = ai;
  }
  __syncthreads();
  if (t < 4) {
    const int comp = t >> 1, part = t & 1;          // u or v, re or im
    // total force coefficients: f_x - (1/2) D t_y ; f_y + (1/2) D t_x
    double a[DP_MAX_NZ + 2], b[DP_MAX_NZ + 2], c[DP_MAX_NZ + 2];
    {
      const double* tq = fc[comp == 0 ? 3 : 2][part];
      double d1 = 0.0, d2 = 0.0;                    // d_{n+1}, d_{n+2}
      for (int n = N; n >= 0; --n) {
        double d = d2 + (n + 1 <= N ? 2.0 * (n + 1) * tq[n + 1] : 0.0);
        double Dt = d / s * (n == 0 ? 0.5 : 1.0);
        double f = fc[comp][part][n] + (comp == 0 ? -0.5 : 0.5) * Dt;
        a[n] = (n <= N - 2) ? -(s * s) * f / A.eta : 0.0;       // a_n = (H/2)^2 r_n, r = -f/eta
        d2 = d1; d1 = d;
      }
      a[N + 1] = 0.0;
    }
    for (int n = 1; n <= N - 1; ++n) b[n] = ((n == 1 ? 2.0 : 1.0) * a[n - 1] - a[n + 1]) / (2.0 * n);
    b[N] = 0.0; b[N + 1] = 0.0; b[0] = 0.0;
    if (A.wall_mode == DP_BOTTOM_WALL) {
      double sb = 0.0;
      for (int n = N - 1; n >= 1; --n) sb += b[n];
      b[0] = -sb;                                                // du/dz(H) = (1/s) sum b_n = 0   (eq 52)
      for (int n = 1; n <= N; ++n) c[n] = ((n == 1 ? 2.0 : 1.0) * b[n - 1] - b[n + 1]) / (2.0 * n);
      double sc = 0.0;
      for (int n = N; n >= 1; --n) sc += (n & 1) ? -c[n] : c[n];
      c[0] = -sc;                                                // u(0) = sum (-1)^n c_n = 0
    } else {
      for (int n = 2; n <= N; ++n) c[n] = (b[n - 1] - b[n + 1]) / (2.0 * n);
      double so = 0.0, se = 0.0;
      for (int n = N; n >= 2; --n) { if (n & 1) so += c[n]; else se += c[n]; }
      c[1] = -so; c[0] = -se;                                    // u(0) = u(H) = 0   ((A12), no slip)
      b[0] = c[1] + 0.5 * b[2];                                  // c_1 = b_0 - b_2/2
    }
    for (int n = 0; n <= N; ++n) { uc[comp][part][n] = c[n]; ub[comp][part][n] = n <= N - 1 ? b[n] / s : 0.0; }
  }
  __syncthreads();
  // synthesis and store: u, v, w = 0; omega_x = -(1/2) dz v, omega_y = +(1/2) dz u, omega_z = 0
  const double scl = 1.0 / ((double)A.nx * (double)A.ny);
  for (int idx = t; idx < nz; idx += blockDim.x) {
    const int l = idx;
    double u[2][2] = {{0, 0}, {0, 0}}, du[2][2] = {{0, 0}, {0, 0}};
    for (int n = 0; n < nz; ++n) {
      const double cs = ct_full[n * nz + l];
      for (int comp = 0; comp < 2; ++comp)
        for (int part = 0; part < 2; ++part) { u[comp][part] += cs * uc[comp][part][n]; du[comp][part] += cs * ub[comp][part][n]; }
    }
    const size_t off = (size_t)l * A.n_slow * A.pitch;
    A.cplx[0 * A.cplx_field + off] = make_double2(u[0][0] * scl, u[0][1] * scl);
    A.cplx[1 * A.cplx_field + off] = make_double2(u[1][0] * scl, u[1][1] * scl);
    A.cplx[2 * A.cplx_field + off] = make_double2(0.0, 0.0);
    if (A.omega) {
      A.cplx[3 * A.cplx_field + off] = make_double2(-0.5 * du[1][0] * scl, -0.5 * du[1][1] * scl);
      A.cplx[4 * A.cplx_field + off] = make_double2(0.5 * du[0][0] * scl, 0.5 * du[0][1] * scl);
      A.cplx[5 * A.cplx_field + off] = make_double2(0.0, 0.0);
    }
  }
}

template <int NZ> size_t solve_smem_bytes() { return sizeof(double) * (size_t)SolveSmem<NZ>::DOUBLES; }

template <int NZ> void host_tables(std::vector<double>& out) {
  typedef long double ld;
  const ld PI = 3.141592653589793238462643383279502884L;
  constexpr int N = NZ - 1, LH = NZ / 2;
  out.assign(Tab<NZ>::SIZE, 0.0);
  for (int n = 0; n <= N; ++n)
    for (int l = 0; l < LH; ++l) out[Tab<NZ>::CA + n * LH + l] = (double)cosl(PI * n * l / N);
  for (int l = 0; l < LH; ++l)
    for (int j = 0; j < LH; ++j) {
      out[Tab<NZ>::SE + l * LH + j] = (double)cosl(PI * (2 * j) * l / N);
      out[Tab<NZ>::SO + l * LH + j] = (double)cosl(PI * (2 * j + 1) * l / N);
    }
  for (int l = 0; l <= N; ++l) out[Tab<NZ>::XI + l] = (double)cosl(PI * l / N);
  // P_n, Q_n: with a = unit vector e_n (n <= N-2), b_m = (cbar_{m-1} a_{m-1} - a_{m+1})/(2m) (1 <= m <= N-1),
  // c_m = (cbar_{m-1} b_{m-1} - b_{m+1})/(2m) (1 <= m <= N), b_0 = 0:  P_n = sum of b_m over m of the other parity,
  // Q_n = sum of c_m over m >= 1 of n's parity.
  for (int n = 0; n <= N - 2; ++n) {
    std::vector<ld> a(NZ + 3, 0), b(NZ + 3, 0), c(NZ + 3, 0);
    a[n] = 1;
    for (int mm = 1; mm <= N - 1; ++mm) b[mm] = ((mm - 1 == 0 ? 2 : 1) * a[mm - 1] - a[mm + 1]) / (2 * (ld)mm);
    for (int mm = 1; mm <= N; ++mm) c[mm] = ((mm - 1 == 0 ? 2 : 1) * b[mm - 1] - b[mm + 1]) / (2 * (ld)mm);
    ld p = 0, q = 0;
    for (int mm = 1; mm <= N; ++mm) { if ((mm - n) % 2 != 0) p += b[mm]; else q += c[mm]; }
    out[Tab<NZ>::P + n] = (double)p; out[Tab<NZ>::Q + n] = (double)q;
  }
}

template <int NZ> cudaError_t set_attr_nz() {      // per device: called by every plan at creation, on its own device
  return cudaFuncSetAttribute(k_solve<NZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)solve_smem_bytes<NZ>());
}

template <int NZ> cudaError_t launch_nz(const SolveArgs& A, cudaStream_t st) {
  const size_t smem = solve_smem_bytes<NZ>();
  dim3 grid((A.n_fast + TM - 1) / TM, A.n_slow);
  k_solve<NZ><<<grid, SOLVE_THREADS, smem, st>>>(A);
  return cudaGetLastError();
}

int nz_slot(int nz) { return nz == 16 ? 0 : nz == 32 ? 1 : nz == 48 ? 2 : -1; }

}  // namespace

bool dp_solve_supports_nz(int nz) { return nz_slot(nz) >= 0; }

cudaError_t dp_solve_upload_tables(dp_plan* P) {
  std::vector<double> t;
  cudaError_t e = cudaSuccess;
  const int nz = P->p.nz;
  if (nz == 16) { host_tables<16>(t); e = cudaMemcpyToSymbol(c_tab16, t.data(), sizeof(double) * t.size()); }
  else if (nz == 32) { host_tables<32>(t); e = cudaMemcpyToSymbol(c_tab32, t.data(), sizeof(double) * t.size()); }
  else if (nz == 48) { host_tables<48>(t); e = cudaMemcpyToSymbol(c_tab48, t.data(), sizeof(double) * t.size()); }
  else return cudaErrorInvalidValue;
  if (e != cudaSuccess) return e;
  if (nz == 16) e = set_attr_nz<16>(); else if (nz == 32) e = set_attr_nz<32>(); else e = set_attr_nz<48>();
  if (e != cudaSuccess) return e;
  if (!P->d_ct_full) {
    typedef long double ld;
    const ld PI = 3.141592653589793238462643383279502884L;
    std::vector<double> ct((size_t)nz * nz);
    for (int n = 0; n < nz; ++n) for (int l = 0; l < nz; ++l) ct[(size_t)n * nz + l] = (double)cosl(PI * n * l / (nz - 1));
    e = cudaMalloc(&P->d_ct_full, sizeof(double) * ct.size());
    if (e != cudaSuccess) return e;
    P->device_bytes += sizeof(double) * ct.size();
    e = cudaMemcpy(P->d_ct_full, ct.data(), sizeof(double) * ct.size(), cudaMemcpyHostToDevice);
  }
  return e;
}

void dp_solve_destroy_tables(dp_plan* P) {
  if (P->d_ct_full) { cudaFree(P->d_ct_full); P->d_ct_full = nullptr; }
}

cudaError_t dp_launch_solve(dp_plan* P, bool with_torque_field, bool want_omega, cudaStream_t st) {
  SolveArgs A;
  A.cplx = P->d_cplx; A.cplx_field = P->cplx_field;
  A.nx = P->p.nx; A.ny = P->p.ny; A.nkx = P->nkx;
  A.n_fast = P->nkx; A.n_slow = P->p.ny; A.pitch = P->nkxp; A.fast_is_x = 1; A.ky_of_pos = nullptr; A.lmin = P->d_lmin;
  if (P->own_fft) { A.n_fast = P->p.ny; A.n_slow = P->nkx; A.pitch = P->p.ny; A.fast_is_x = 0; A.ky_of_pos = dp_fft_own_ky_table(P); }
  A.Lx = P->p.Lx; A.Ly = P->p.Ly; A.H = P->p.H; A.eta = P->p.eta;
  A.wall_mode = P->p.wall_mode; A.torque = with_torque_field ? 1 : 0; A.omega = want_omega ? 1 : 0;
  cudaError_t e;
  switch (P->p.nz) {
    case 16: e = launch_nz<16>(A, st); break;
    case 32: e = launch_nz<32>(A, st); break;
    case 48: e = launch_nz<48>(A, st); break;
    default: return cudaErrorInvalidValue;
  }
  if (e != cudaSuccess) return e;
  k_zero_mode<<<1, 64, 0, st>>>(A, P->p.nz, P->d_ct_full);
  return cudaGetLastError();
}
