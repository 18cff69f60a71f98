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
// B200 mapping: one CTA = 16 consecutive modes of one row of the half spectrum, 6 warps, 4 CTAs per SM at nz = 32.
// A complex column of the tile is a [nz][32] array of doubles in shared memory: row n = Chebyshev index (or node), the 32
// entries of a row are (mode, re/im) = "lane" 2*mode + part, stored at position lane ^ swz(n) (an XOR swizzle of the
// 4-lane groups of a row, see swz()).  Two kinds of work run on this layout:
//  * the Chebyshev transforms are dense matrix products (cosine table x 32 columns): they run on the fp64 tensor pipe as
//    mma.sync m8n8k4 (SASS DMMA), folded by the symmetry cos(n (N-l) pi/N) = (-1)^n cos(n l pi/N) into two half-size
//    products per column; the table fragments come from a small per-plan global table (L1 resident), the data fragments
//    straight from the swizzled tile (conflict free), 8 columns ("block") at a time so that a column's four blocks can go to
//    different warps;
//  * everything else (z-derivative recurrences, tridiagonal sweeps, boundary functionals, the correction) acts on a lane's
//    own column only; the imaginary unit couples a lane to its neighbour (lane ^ 1), a shuffle or a neighbouring address.
// Five columns live in shared memory: f_x -> u, f_y -> v, f_z -> f_z - dz p -> w, t_x -> p -> dz u, t_y -> (E, zE) -> dz v.
// Their rows are stored split by parity (see crow()), which makes each folded transform a square product in place on half the
// rows and lets a warp keep the table fragments in registers while it walks over the column blocks of a tile.
#include <cmath>
#include <vector>

#include "solve_common.cuh"

using namespace dp_solve;

namespace {

constexpr int SOLVE_WARPS = 6;
constexpr int SOLVE_THREADS = SOLVE_WARPS * 32;

// ---- shared-memory swizzle: element (row n, lane c) of a column tile lives at n * LN + (c ^ swz(n)).
// swz(n) is 0, 4, 8 or 12 (it permutes the four 4-lane groups inside each half of a row and keeps (re, im) pairs adjacent),
// chosen so that the DMMA fragment accesses are bank-conflict free: it is injective on every aligned group of four consecutive
// rows and on {8m + 2k + p, k < 4}, and rows n, n+1 (n even) and n, n+2 (n = 0, 1 mod 4) differ in its upper bit.
__host__ __device__ constexpr int swz(int n) { return ((((n ^ (n >> 1)) & 1) << 1) | (((n >> 1) ^ (n >> 2)) & 1)) << 2; }
// Rows of a tile are "parity split": with NP = ceil(nz/2),
//   nodal side:        e_l = g_l + g_{N-l} at row l (l < NP; the middle node of an odd nz alone), o_l = g_l - g_{N-l} at row NP + l;
//   coefficient side:  g^_n at row n/2 for even n, at row NP + (n-1)/2 for odd n.
// The folded cosine transforms map rows [0, NP) to rows [0, NP) and rows [NP, nz) to rows [NP, nz): each is in place on its
// own rows and the two never touch the same data.
template <int NZ> __host__ __device__ constexpr int crow(int n) { return (n & 1) ? (NZ + 1) / 2 + (n >> 1) : (n >> 1); }
#define EL(tile, n, ln) (tile)[crow<NZ>(n) * LN + ((ln) ^ swz(crow<NZ>(n)))]

// ---- constant tables per compiled nz: P[n], Q[n] = boundary-row functionals of a unit a_n (see chain()), XI[l] = cos(l pi/N)
template <int NZ> struct Tab { static constexpr int P = 0, Q = NZ, XI = 2 * NZ, SIZE = 3 * NZ; };
#define DP_SOLVE_NZ_LIST(X) X(16) X(19) X(24) X(26) X(32) X(40) X(48) X(64)
template <int NZ> __device__ __forceinline__ const double* tab();
#define X(NZ) __constant__ double c_tab##NZ[Tab<NZ>::SIZE]; \
  template <> __device__ __forceinline__ const double* tab<NZ>() { return c_tab##NZ; }
DP_SOLVE_NZ_LIST(X)
#undef X

// ---- geometry of the folded transforms: NP pairs (l, N-l) of nodes (the middle node pairs with itself when nz is odd),
// even coefficients n = 2j and odd coefficients n = 2j+1, all padded to LP = a multiple of 8; KB k-blocks of 4, MB m-blocks of 8.
// Fragment table (global, per plan): [4 kinds][MB][KB][32 lanes]; kind 0, 1: analysis even / odd, 2, 3: synthesis even / odd.
template <int NZ> struct Tr {
  static constexpr int NP = (NZ + 1) / 2, LP = (NP + 7) / 8 * 8, KB = LP / 4, MB = LP / 8, FRAGS = 4 * MB * KB;
};



// D(8x8) += A(8x4) B(4x8) on the fp64 tensor pipe: lane t holds A[t/4][t%4], B[t%4][t/4], D[t/4][2(t%4)], D[t/4][2(t%4)+1]
__device__ __forceinline__ void dmma(double (&d)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}
__device__ __forceinline__ int swz_rt(int n) { return ((((n ^ (n >> 1)) & 1) << 1) | (((n >> 1) ^ (n >> 2)) & 1)) << 2; }

// ---- one folded cosine transform of one parity, on the fp64 tensor pipe (one warp), in place on that parity's rows:
//   analysis (kind 0 even, 1 odd):  g^_n = (2/N)(1/c~_n) sum_{l < NP} (1/c~_l) cos(n l pi/N) {e_l | o_l}   (n even | odd),
//     which is the DCT-I  g^_n = (2/N)(1/c~_n) sum_l (1/c~_l) g_l cos(n l pi/N)  folded with cos(n (N-l) pi/N) = (-1)^n cos(n l pi/N);
//   synthesis (kind 2 even, 3 odd): E_l = sum_j g^_{2j} cos(2j l pi/N) | O_l = sum_j g^_{2j+1} cos((2j+1) l pi/N), so that
//     g_l = E_l + O_l, g_{N-l} = E_l - O_l.
//   NBI 8-column blocks nb0 .. are transformed with the table fragments (all weights are in the table) held in registers.
template <int NZ, int NBI>
__device__ __forceinline__ void transform_item(double* __restrict__ tile, int kind, int nb0, const double* __restrict__ frag, int lane) {
  typedef Tr<NZ> G;
  constexpr int NP = G::NP, KB = G::KB, MB = G::MB;
  const int g = lane >> 2, t = lane & 3;
  const int par = kind & 1;
  const int row0 = par ? NP : 0, cnt = par ? NZ - NP : NP;
  const double* __restrict__ fk = frag + (size_t)(kind * MB) * KB * 32 + lane;
  constexpr bool FRAG_REGS = MB * KB <= 8;  // larger tables are re-read from L1 per block
  double fa[FRAG_REGS ? MB : 1][FRAG_REGS ? KB : 1];
  if (FRAG_REGS) {
#pragma unroll
    for (int mb = 0; mb < MB; ++mb)
#pragma unroll
      for (int kb = 0; kb < KB; ++kb) fa[FRAG_REGS ? mb : 0][FRAG_REGS ? kb : 0] = __ldg(fk + (mb * KB + kb) * 32);
  }
  int xo[KB];                                // offsets of this lane's operand rows, swizzle included (column block 0)
#pragma unroll
  for (int kb = 0; kb < KB; ++kb) { const int r = row0 + kb * 4 + t; xo[kb] = r * LN + (g ^ swz_rt(r)); }
#pragma unroll
  for (int nbi = 0; nbi < NBI; ++nbi) {
    const int nb = nb0 + nbi;
    double x[KB];
#pragma unroll
    for (int kb = 0; kb < KB; ++kb) x[kb] = (kb * 4 + t < cnt) ? tile[xo[kb] ^ (nb * 8)] : 0.0;
    double acc[MB][2];
#pragma unroll
    for (int mb = 0; mb < MB; ++mb) acc[mb][0] = acc[mb][1] = 0.0;
#pragma unroll
    for (int kb = 0; kb < KB; ++kb)
#pragma unroll
      for (int mb = 0; mb < MB; ++mb) dmma(acc[mb], FRAG_REGS ? fa[FRAG_REGS ? mb : 0][FRAG_REGS ? kb : 0] : __ldg(fk + (mb * KB + kb) * 32), x[kb]);
    __syncwarp();                            // every lane has read its operands of this block before the block is overwritten
#pragma unroll
    for (int mb = 0; mb < MB; ++mb) {
      const int m = mb * 8 + g, r = row0 + m;
      if (m < cnt) *reinterpret_cast<double2*>(&tile[r * LN + ((nb * 8 + 2 * t) ^ swz_rt(r))]) = make_double2(acc[mb][0], acc[mb][1]);
    }
  }
}


// ---- coefficient-space z-derivative of a lane's column (both parities), top-down recurrence
//   d_N = 0, d_n = d_{n+2} + 2(n+1) g_{n+1},  (D g)_n = (2/H) d_n (d_0 halved);  dst[n] (+)= scale * (D src)_n
template <int NZ, bool ACC> __device__ __forceinline__ void deriv_column(const double* __restrict__ src, double* __restrict__ dst, int lane, double inv_s, double scale) {
  constexpr int N = NZ - 1;
  double g[NZ];
#pragma unroll
  for (int n = 1; n <= N; ++n) g[n] = EL(src, n, lane);
  double d0 = 0.0, d1 = 0.0;          // running sums of the two parities
  const double f = inv_s * scale;
#pragma unroll
  for (int n = N; n >= 0; --n) {
    double& d = (n & 1) ? d1 : d0;
    if (n + 1 <= N) d = fma(2.0 * (n + 1), g[n + 1], d);
    const double val = d * (n == 0 ? 0.5 * f : f);
    if (ACC) EL(dst, n, lane) += val; else EL(dst, n, lane) = val;
  }
}


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
//      Writes y's coefficients c_n of parity PAR to tile `col` and, if SUB_D, SUBTRACTS the coefficients of dy/dz (they have the
//      OTHER parity) from tile `dcol`.  Returns S_c = sum of the c_n written (incl. c_0 for the even chain).
template <int NZ, int PAR>
__device__ __forceinline__ double chain(bool SUB_D, double (&a)[Ch<NZ, PAR>::NR], double rho0, const double* __restrict__ Fm, const double* __restrict__ Fi,
                                        const double* __restrict__ Fa, double* __restrict__ col, double* __restrict__ dcol, int lane, double k,
                                        double k2, double inv_s, double beta_bc, double invBg, double* __restrict__ sum_b) {
  constexpr int N = NZ - 1, n0 = Ch<NZ, PAR>::n0, NR = Ch<NZ, PAR>::NR;
  const double* __restrict__ T = tab<NZ>();
  if (!PAR) a[0] = fma(0.25 * k2, rho0, a[0]);               // even chain: row 2 carries (kappa^2/4) rho_0
#pragma unroll
  for (int j = 1; j < NR; ++j) a[j] = fma(-Fm[(n0 + 2 * j) * TM], a[j - 1], a[j]);
  double SP = 0.0, SQ = 0.0, next = 0.0;
#pragma unroll
  for (int j = NR - 1; j >= 0; --j) {
    const int n = n0 + 2 * j;
    const double v = (a[j] - row_u<NZ>(n, k2) * next) * Fi[n * TM];
    a[j] = v; next = v;
    SP = fma(T[Tab<NZ>::P + n], v, SP); SQ = fma(T[Tab<NZ>::Q + n], v, SQ);
  }
  if (!PAR) { SP = fma(T[Tab<NZ>::P + 0], rho0, SP); SQ = fma(T[Tab<NZ>::Q + 0], rho0, SQ); }
  const double border = (beta_bc - (inv_s * SP + k * SQ)) * invBg;       // c_0 (even chain) or b_0 (odd chain)
#pragma unroll
  for (int j = 0; j < NR; ++j) a[j] = fma(border, Fa[(n0 + 2 * j) * TM], a[j]);
  // integrate twice:  b_{n+1} = (cbar_n a_n - a_{n+2}) / (2(n+1)),  c_n = (cbar_{n-1} b_{n-1} - b_{n+1}) / (2n)
  double Sc0 = 0.0, Sc1 = 0.0, bprev;
  double Sb = PAR ? border : 0.0;            // sum of the b_m this chain produces (m of the other parity): (H/2) dy/dz summed (footnote 46)
  if (!PAR) { EL(col, 0, lane) = border; Sc0 = border; bprev = 0.0; }
  else { bprev = border; if (SUB_D) EL(dcol, 0, lane) -= border * inv_s; }
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
      EL(col, n, lane) = c;
      if (i & 1) Sc1 += c; else Sc0 += c;
    }
    if (SUB_D && n + 1 <= N - 1) EL(dcol, n + 1, lane) -= bn1 * inv_s;
    if (sum_b && n + 1 <= N - 1) Sb += bn1;
    bprev = bn1;
  }
  if (sum_b) *sum_b = Sb;
  return Sc0 + Sc1;
}



// ---- one BVP item of a lane: kind 0 = pressure (eqs 15, 17): right-hand side i k.f + dz f_z, p -> tile 3, and f_z -= dz p in
//      tile 2; kind 1 = u or v (comp 0, 1), kind 2 = w (eq 18 with BCs 22, 24): f_c (tile comp) is overwritten by u_c.
//      One code path per parity so that the chain sweeps exist once in the instruction stream.
template <int NZ, int PAR>
__device__ __noinline__ double bvp_item(int kind, int comp, double* __restrict__ C, const double* __restrict__ F, int lane, int mode, ModeK K,
                                        double s, double inv_s, double eta, double invBg, double pH_own, double p0_own, double pH_oth, double p0_oth,
                                        double* __restrict__ sum_b) {
  constexpr int N = NZ - 1, n0 = Ch<NZ, PAR>::n0, NR = Ch<NZ, PAR>::NR, VS = NZ * LN;
  double a[NR], rho0 = 0.0, beta_bc = 0.0;
  double* col;
  if (kind == 0) {
    const double* fx = C + 0 * VS;                        // read at lane ^ 1: i k f mixes re and im
    const double* fy = C + 1 * VS;
    const double* fz = C + 2 * VS;
    double d = 0.0;
    constexpr int ntop = ((N - PAR) & 1) ? N - 1 : N;     // largest n <= N with parity PAR
    const double s2 = s * s;
#pragma unroll
    for (int i = 0; i <= ntop / 2; ++i) {
      const int n = ntop - 2 * i;
      if (n < 0) break;
      if (n + 1 <= N) d = fma(2.0 * (n + 1), EL(fz, n + 1, lane), d);
      if (n <= N - 2) {
        const double r = fma(K.sgI, fma(K.kxt, EL(fx, n, lane ^ 1), K.kyt * EL(fy, n, lane ^ 1)), d * (n == 0 ? 0.5 * inv_s : inv_s)) * s2;
        if (n >= n0) a[n >= n0 ? (n - n0) / 2 : 0] = r; else rho0 = r;
      }
    }
    col = C + 3 * VS;
  } else {
    col = C + comp * VS;
    const double sc = s * s / eta;
    double gH, g0;
    const double kc = comp == 0 ? K.kxt : K.kyt;
    if (kind == 1) {
      // r = (i k_c p - f_c)/eta ; (dz + k) u(H) = -(i k_c/(2 k eta)) p(H) ; (dz - k) u(0) = +(i k_c/(2 k eta)) p(0)      (eqs 18, 22)
      const double* p = C + 3 * VS;
      const double f = K.sgI * kc;
#pragma unroll
      for (int i = 0; i <= (N - 2 - PAR) / 2; ++i) {
        const int n = PAR + 2 * i;
        const double r = (f * EL(p, n, lane ^ 1) - EL(col, n, lane)) * sc;
        if (n >= n0) a[n >= n0 ? (n - n0) / 2 : 0] = r; else rho0 = r;
      }
      const double c = kc / (2.0 * K.k * eta);
      gH = -K.sgI * c * pH_oth; g0 = K.sgI * c * p0_oth;
    } else {
      // r = (dz p - f_z)/eta = -(f_z - dz p)/eta ; (dz + k) w(H) = p(H)/(2 eta) ; (dz - k) w(0) = p(0)/(2 eta)          (eqs 18, 24)
#pragma unroll
      for (int i = 0; i <= (N - 2 - PAR) / 2; ++i) {
        const int n = PAR + 2 * i;
        const double r = -EL(col, n, lane) * sc;
        if (n >= n0) a[n >= n0 ? (n - n0) / 2 : 0] = r; else rho0 = r;
      }
      gH = pH_own / (2.0 * eta); g0 = p0_own / (2.0 * eta);
    }
    beta_bc = PAR ? 0.5 * (gH + g0) : 0.5 * (gH - g0);
  }
  return chain<NZ, PAR>(kind == 0, a, rho0, F + 0 * NZ * TM + mode, F + 1 * NZ * TM + mode, F + 2 * NZ * TM + mode, col, C + 2 * VS, lane,
                        K.k, K.k2, inv_s, beta_bc, invBg, sum_b);
}


template <int NZ> struct SolveSmem {
  static constexpr int VS = NZ * LN;                                   // one complex column tile [n][lane ^ swz(n)]
  static constexpr int COLS = 5 * VS;                                  // tiles 0..4
  static constexpr int FACT = COLS;                                    // [3][NZ][TM]: multipliers, inverse pivots, border solution
  static constexpr int IBG = FACT + 3 * NZ * TM;                       // [2][TM] 1/B_g of the even / odd chain
  static constexpr int SUM = IBG + 2 * TM;                             // [4][2][LN] S_c of (p,u,v,w) x (even, odd chain)
  static constexpr int SUMB = SUM + 8 * LN;                            // [2][2][LN] S_b of (u,v) x (even, odd chain): wall derivatives (partial slip)
  static constexpr int DOUBLES = SUMB + 4 * LN;
  static constexpr int CORR = FACT;                                    // [12][LN] slit correction coefficients: the factors are dead by then
  static_assert(12 * LN <= 3 * NZ * TM, "correction coefficients fit in the factor area");
  static constexpr int PER_SM = (227 * 1024) / (DOUBLES * 8 + 1024);   // CTAs that fit an SM's shared memory
  static constexpr int CTAS = PER_SM >= 4 ? 4 : (PER_SM >= 1 ? PER_SM : 1);
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
__global__ void __launch_bounds__(SOLVE_THREADS, SolveSmem<NZ>::CTAS) k_solve(SolveArgs A) {
  extern __shared__ __align__(16) double smem[];
  constexpr int VS = NZ * LN;
  typedef SolveSmem<NZ> S;
  double* C = smem;                      // tiles: 0 f_x->u, 1 f_y->v, 2 f_z->f_z - dz p->w, 3 t_x->p->dz u, 4 t_y->(E, zE)->dz v
  double* F = smem + S::FACT;
  double* s_ibg = smem + S::IBG;
  double* s_sum = smem + S::SUM;
  double* s_sumb = smem + S::SUMB;
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

  // ---------------- phase 0: the nodal columns go HBM -> shared memory as 16-byte cp.async (one (re, im) pair per copy, L1
  // bypassed, no registers).  A warp takes the node pairs (l, N-l), l = wid, wid + 6, ... < NP: node l lands in row l, node N-l in
  // row NP + l; its lanes 0-15 copy the modes of tiles 0, 2, 4, its lanes 16-31 those of tiles 1, 3.  t_z is only needed for the
  // fold below and travels through registers.  While the loads fly, warps 0, 1 factor the two chains.  Then every warp, for the
  // pairs it loaded itself, folds the algebraic part of (1/2) curl t into f (eq 7) and replaces (g_l, g_{N-l}) by (e_l, o_l).
  typedef Tr<NZ> G;
  constexpr int N = NZ - 1, NP = G::NP;
  constexpr int PAIRS = (NP + SOLVE_WARPS - 1) / SOLVE_WARPS;
  const int lm = __ldg(A.lmin);
  double tz[PAIRS][2];
  {
    const int sub = lane >> 4, m = lane & 15;
    const int mfast = blockIdx.x * TM + m;
    const bool mvalid = mfast < A.n_fast;
    const size_t moff = (size_t)islow * A.pitch + mfast;
    const int ntile = A.torque ? 5 : 3;
#pragma unroll
    for (int r = 0; r < PAIRS; ++r) {
      const int lp = wid + r * SOLVE_WARPS;
      tz[r][0] = tz[r][1] = 0.0;
      if (lp < NP) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int l = h ? N - lp : lp, row = h ? NP + lp : lp;          // node, row
          if (h && l == lp) continue;                                     // the middle node of an odd nz has no partner
          const int sw = swz_rt(row);
          const bool live = mvalid && l >= lm;
#pragma unroll
          for (int q = 0; q < 3; ++q) {
            const int c = 2 * q + sub;
            if (c < ntile) {
              double* dst = &C[c * VS + row * LN + ((2 * m) ^ sw)];
              if (live) cp_async16(dst, A.cplx + c * A.cplx_field + l * plane + moff);
              else *reinterpret_cast<double2*>(dst) = make_double2(0.0, 0.0);
            }
          }
          if (A.torque && valid && l >= lm) tz[r][h] = ldg_stream(&gin[2 * (5 * A.cplx_field + l * plane + off0) + part]);
        }
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
  }
  TMARK(2);
  cp_async_wait_all();
  __syncwarp();
  {
    const int ntile = A.torque ? 5 : 3;
#pragma unroll
    for (int r = 0; r < PAIRS; ++r) {
      const int lp = wid + r * SOLVE_WARPS;
      if (lp < NP) {
        const bool pair = (N - lp) != lp;
        const int ra = lp, rb = NP + lp;
        const int oa = ra * LN + (lane ^ swz_rt(ra)), ob = rb * LN + (lane ^ swz_rt(rb));
        double va[5], vb[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) { va[c] = vb[c] = 0.0; if (c < ntile) { va[c] = C[c * VS + oa]; if (pair) vb[c] = C[c * VS + ob]; } }
        if (A.torque) {
          // the OTHER part of t: i k x t mixes re and im
          const double txa = __shfl_xor_sync(0xffffffffu, va[3], 1), tya = __shfl_xor_sync(0xffffffffu, va[4], 1), tza = __shfl_xor_sync(0xffffffffu, tz[r][0], 1);
          const double txb = __shfl_xor_sync(0xffffffffu, vb[3], 1), tyb = __shfl_xor_sync(0xffffffffu, vb[4], 1), tzb = __shfl_xor_sync(0xffffffffu, tz[r][1], 1);
          va[0] = fma(0.5 * K.sgI * K.kyt, tza, va[0]);                        // f_x += (1/2) i k_y t_z
          va[1] = fma(-0.5 * K.sgI * K.kxt, tza, va[1]);                       // f_y -= (1/2) i k_x t_z
          va[2] = fma(0.5 * K.sgI, K.kxt * tya - K.kyt * txa, va[2]);          // f_z += (1/2) i (k_x t_y - k_y t_x)
          vb[0] = fma(0.5 * K.sgI * K.kyt, tzb, vb[0]);
          vb[1] = fma(-0.5 * K.sgI * K.kxt, tzb, vb[1]);
          vb[2] = fma(0.5 * K.sgI, K.kxt * tyb - K.kyt * txb, vb[2]);
        }
#pragma unroll
        for (int c = 0; c < 5; ++c)
          if (c < ntile) { C[c * VS + oa] = va[c] + vb[c]; if (pair) C[c * VS + ob] = va[c] - vb[c]; }
      }
    }
  }
  TMARK(3);
  __syncthreads();

  // ---------------- phase 1: Chebyshev analysis of f_x, f_y, f_z [, t_x, t_y] on the tensor pipe, one (tile, parity) item per warp   (step 2)
  {
    const int nitems = (A.torque ? 5 : 3) * 2;
    for (int i = wid; i < nitems; i += SOLVE_WARPS) transform_item<NZ, 4>(C + (i >> 1) * VS, i & 1, 0, A.frag, lane);
  }
  TMARK(4);
  __syncthreads();

  // ---------------- phases 2, 3: warps 0, 1: f_x -= (1/2) D t_y, f_y += (1/2) D t_x (eq 7), then the pressure BVP (eqs 15, 17), one
  // chain each.  Warps 2-5 meanwhile evaluate e^{-k z_l} and z_l e^{-k z_l} at the nodes, put them into tile 4 once t_y has
  // been consumed, and transform them (one 8-lane block each); their coefficients are needed for the correction (step 6).
  if (wid < 2) {
    if (A.torque) deriv_column<NZ, true>(C + (wid == 0 ? 4 : 3) * VS, C + wid * VS, lane, inv_s, wid == 0 ? -0.5 : 0.5);
    TMARK(5);
    named_arrive(2, SOLVE_THREADS);                        // t_y has been read: tile 4 may be overwritten
    named_sync(1, 64);                                     // f_x and f_y are complete (and t_x consumed) before either chain starts
    double Sc;
    if (wid) Sc = bvp_item<NZ, 1>(0, 0, C, F, lane, mode, K, s, inv_s, eta, s_ibg[TM + mode], 0.0, 0.0, 0.0, 0.0, nullptr);
    else Sc = bvp_item<NZ, 0>(0, 0, C, F, lane, mode, K, s, inv_s, eta, s_ibg[mode], 0.0, 0.0, 0.0, 0.0, nullptr);
    s_sum[(0 * 2 + wid) * LN + lane] = Sc;
  } else {
    constexpr int ER = (NP + 3) / 4;                       // node pairs (l, N-l) per thread
    double ee[ER], eo[ER];
#pragma unroll
    for (int r = 0; r < ER; ++r) {
      const int lp = (wid - 2) + 4 * r;
      ee[r] = eo[r] = 0.0;
      if (lp < NP) {
        const double za = s * (1.0 + T[Tab<NZ>::XI + lp]);
        const double Ea = exp(-K.k * za);
        const double a = part ? za * Ea : Ea;
        double b = 0.0;
        if (N - lp != lp) {
          const double zb = s * (1.0 + T[Tab<NZ>::XI + N - lp]);
          const double Eb = exp(-K.k * zb);
          b = part ? zb * Eb : Eb;
        }
        ee[r] = a + b; eo[r] = a - b;
      }
    }
    named_sync(2, SOLVE_THREADS);
#pragma unroll
    for (int r = 0; r < ER; ++r) {
      const int lp = (wid - 2) + 4 * r;
      if (lp < NP) {
        C[4 * VS + lp * LN + (lane ^ swz_rt(lp))] = ee[r];
        if (N - lp != lp) C[4 * VS + (NP + lp) * LN + (lane ^ swz_rt(NP + lp))] = eo[r];
      }
    }
    named_sync(3, 128);
    transform_item<NZ, 2>(C + 4 * VS, (wid - 2) & 1, ((wid - 2) >> 1) * 2, A.frag, lane);
  }
  TMARK(6);
  __syncthreads();

  // ---------------- phase 4: the velocity BVPs (eq 18) with BCs (22), (24), one warp per (component, chain)
  {
    const int comp = wid >> 1, par = wid & 1;
    const int kind = comp == 2 ? 2 : 1;
    const double se = s_sum[0 * LN + lane], so = s_sum[1 * LN + lane];
    const double pH = se + so, p0 = se - so;              // p(H) = sum p_n, p(0) = sum (-1)^n p_n  ("direct summation")
    const double pHo = __shfl_xor_sync(0xffffffffu, pH, 1), p0o = __shfl_xor_sync(0xffffffffu, p0, 1);
    double Sc, Sb = 0.0;
    double* want_sb = (A.slip && comp < 2) ? &Sb : nullptr;        // partial slip needs du/dz, dv/dz of the DP solution on the walls
    if (par) Sc = bvp_item<NZ, 1>(kind, comp, C, F, lane, mode, K, s, inv_s, eta, s_ibg[TM + mode], pH, p0, pHo, p0o, want_sb);
    else Sc = bvp_item<NZ, 0>(kind, comp, C, F, lane, mode, K, s, inv_s, eta, s_ibg[mode], pH, p0, pHo, p0o, want_sb);
    s_sum[((1 + comp) * 2 + par) * LN + lane] = Sc;
    if (want_sb) s_sumb[(comp * 2 + par) * LN + lane] = Sb;
  }
  TMARK(7);
  __syncthreads();

  // ---------------- phase 5: correction coefficients (bottom wall: every warp for itself; slit: warp 0, shared)
  double cf[3][4];
  double ssum[6], ssb[4];
#pragma unroll
  for (int i = 0; i < 6; ++i) ssum[i] = s_sum[(2 + i) * LN + lane];
#pragma unroll
  for (int i = 0; i < 4; ++i) ssb[i] = A.slip ? s_sumb[i * LN + lane] : 0.0;
  if (A.wall_mode == DP_BOTTOM_WALL) {
    correction_coefficients(ssum, ssb, K, A.H, DP_BOTTOM_WALL, 0.0, 0.0, cf);
  } else {
    if (wid == 0) {
      correction_coefficients(ssum, ssb, K, A.H, DP_SLIT, A.l0, A.lH, cf);
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
  // (rows [0, NP) hold the even coefficients, rows [NP, nz) the odd ones)
  for (int r = wid; r < NZ; r += SOLVE_WARPS) {
    const int sw = swz_rt(r);
    const double mine = C[4 * VS + r * LN + (lane ^ sw)], other = C[4 * VS + r * LN + ((lane ^ 1) ^ sw)];
    const double en = part ? other : mine, zen = part ? mine : other;
    const double sgn = (r >= NP) ? -1.0 : 1.0;
    const double b2 = sgn * (A.H * en - zen), b3 = sgn * en;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double add = fma(cf[c][0], zen, cf[c][1] * en);
      if (A.wall_mode == DP_SLIT) add = fma(cf[c][2], b2, fma(cf[c][3], b3, add));
      C[c * VS + r * LN + (lane ^ sw)] += add;
    }
  }
  TMARK(8);
  __syncthreads();

  // ---------------- phase 7: dz u, dz v of the TOTAL in coefficient space (reading G12) -> tiles 3, 4 (warps 0, 1) while warps 2-5
  // bring w back to the nodes; then synthesis of u, v [, dz u, dz v], (tile, parity, half) items dealt to the warps
  if (A.omega) {
    if (wid < 2) deriv_column<NZ, false>(C + wid * VS, C + (3 + wid) * VS, lane, inv_s, 1.0);
    else transform_item<NZ, 2>(C + 2 * VS, 2 + ((wid - 2) & 1), ((wid - 2) >> 1) * 2, A.frag, lane);
    TMARK(9);
    __syncthreads();
    for (int i = wid; i < 16; i += SOLVE_WARPS) { const int c = i >> 2; transform_item<NZ, 2>(C + (c < 2 ? c : c + 1) * VS, 2 + (i & 1), (i & 2), A.frag, lane); }
  } else {
    for (int i = wid; i < 6; i += SOLVE_WARPS) transform_item<NZ, 4>(C + (i >> 1) * VS, 2 + (i & 1), 0, A.frag, lane);
  }
  TMARK(10);
  __syncthreads();

  // ---------------- phase 8: back to the nodes g_l = E_l + O_l, g_{N-l} = E_l - O_l; (1/2) curl u (eq 11); scale by 1/(nx ny)
  // for the unnormalised inverse FFT; store
  const double scl = 1.0 / ((double)A.nx * (double)A.ny);
  double* gout = reinterpret_cast<double*>(A.cplx);
  for (int lp = wid; lp < NP; lp += SOLVE_WARPS) {
    const bool pair = (N - lp) != lp;
    const int oa = lp * LN + (lane ^ swz_rt(lp)), ob = (NP + lp) * LN + (lane ^ swz_rt(NP + lp));
    const int nt = A.omega ? 5 : 3;
    double vE[5], vO[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) { vE[c] = vO[c] = 0.0; if (c < nt) { vE[c] = C[c * VS + oa]; if (pair) vO[c] = C[c * VS + ob]; } }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      if (h && !pair) continue;
      const int l = h ? N - lp : lp;
      const double u = h ? vE[0] - vO[0] : vE[0] + vO[0], v = h ? vE[1] - vO[1] : vE[1] + vO[1], w = h ? vE[2] - vO[2] : vE[2] + vO[2];
      double om[3] = {0, 0, 0};
      if (A.omega) {
        const double du = h ? vE[3] - vO[3] : vE[3] + vO[3], dv = h ? vE[4] - vO[4] : vE[4] + vO[4];
        const double uo = __shfl_xor_sync(0xffffffffu, u, 1), vo = __shfl_xor_sync(0xffffffffu, v, 1), wo = __shfl_xor_sync(0xffffffffu, w, 1);
        om[0] = 0.5 * (K.sgI * K.kyt * wo - dv);                          // (1/2)(i k_y w - dz v)
        om[1] = 0.5 * (du - K.sgI * K.kxt * wo);                          // (1/2)(dz u - i k_x w)
        om[2] = 0.5 * K.sgI * (K.kxt * vo - K.kyt * uo);                  // (1/2)(i k_x v - i k_y u)
      }
      if (valid && !zero_mode && l >= lm) {                // planes above every footprint are never interpolated from: not stored
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
//   w = 0;  u'' = -f_x/eta, v'' = -f_y/eta with u(0) = u_wall and (bottom wall) u'(H) = 0, or (slit, (A12)) u(0) - l0 u'(0) = u_wall_0,
//   u(H) + lH u'(H) = u_wall_H (uniform wall velocities; slip lengths l0, lH).
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
    // the unnormalised xy DFT of a uniform wall velocity U is nx ny U at k = 0 (real), and nothing at any other wavenumber
    const double Uw0 = part ? 0.0 : (double)A.nx * (double)A.ny * A.uw0[comp];
    const double UwH = part ? 0.0 : (double)A.nx * (double)A.ny * A.uwH[comp];
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
      c[0] = Uw0 - sc;                                           // u(0) = sum (-1)^n c_n = u_wall (eqs 46, 52; 0 for a wall at rest)
    } else {
      for (int n = 2; n <= N; ++n) c[n] = (b[n - 1] - b[n + 1]) / (2.0 * n);
      double so = 0.0, se = 0.0, sbH = 0.0, sb0 = 0.0;
      for (int n = N; n >= 2; --n) { if (n & 1) so += c[n]; else se += c[n]; }
      for (int n = N - 1; n >= 1; --n) { sbH += b[n]; sb0 += (n & 1) ? -b[n] : b[n]; }
      // (A12): u(H) + lH u'(H) = U_H, u(0) - l0 u'(0) = U_0 with u' = (1/s) sum b_n, b_0 = c_1 + b_2/2:
      //   c_0 + c_1 (1 + lH/s) = T,   c_0 - c_1 (1 + l0/s) = B
      const double rH = A.lH / s, r0 = A.l0 / s;
      const double Tt = UwH - se - so - rH * (0.5 * b[2] + sbH);
      const double Bb = Uw0 - se + so + r0 * (0.5 * b[2] + sb0);
      c[1] = (Tt - Bb) / (2.0 + rH + r0);
      c[0] = Tt - c[1] * (1.0 + rH);
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

// P_n, Q_n, XI_l of the constant table, and the transform fragment table of Tr<NZ>
template <int NZ> void host_tables(std::vector<double>& ctab, std::vector<double>& frag) {
  typedef long double ld;
  const ld PI = 3.141592653589793238462643383279502884L;
  constexpr int N = NZ - 1;
  ctab.assign(Tab<NZ>::SIZE, 0.0);
  for (int l = 0; l <= N; ++l) ctab[Tab<NZ>::XI + l] = (double)cosl(PI * l / N);
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
    ctab[Tab<NZ>::P + n] = (double)p; ctab[Tab<NZ>::Q + n] = (double)q;
  }
  // fragments: lane t of fragment (kind, mb, kb) holds M_kind[mb*8 + t/4][kb*4 + t%4]
  typedef Tr<NZ> G;
  frag.assign((size_t)G::FRAGS * 32, 0.0);
  auto ctil = [&](int i) { return (i == 0 || i == N) ? (ld)2 : (ld)1; };
  for (int kind = 0; kind < 4; ++kind)
    for (int mb = 0; mb < G::MB; ++mb)
      for (int kb = 0; kb < G::KB; ++kb)
        for (int t = 0; t < 32; ++t) {
          const int row = mb * 8 + t / 4, col = kb * 4 + t % 4;
          ld v = 0;
          if (kind < 2) {                // analysis: row = coefficient index j (n = 2j + kind), col = node pair l
            const int n = 2 * row + kind, l = col;
            if (n <= N && l < G::NP) v = (2 / (ld)N) / (ctil(n) * ctil(l)) * cosl(PI * (ld)n * l / N);
          } else {                       // synthesis: row = node l, col = coefficient index j (n = 2j + kind - 2)
            const int l = row, n = 2 * col + (kind - 2);
            if (n <= N && l < G::NP) v = cosl(PI * (ld)n * l / N);
          }
          frag[((size_t)(kind * G::MB + mb) * G::KB + kb) * 32 + t] = (double)v;
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

}  // namespace

bool dp_solve_supports_nz(int nz) {
#define X(NZ) if (nz == NZ) return true;
  DP_SOLVE_NZ_LIST(X)
#undef X
  return false;
}

int dp_solve_nz_list(int* out, int cap) {
  int n = 0;
#define X(NZ) { if (n < cap) out[n] = NZ; ++n; }
  DP_SOLVE_NZ_LIST(X)
#undef X
  return n;
}

cudaError_t dp_launch_solve_pair(dp_plan* P, const SolveArgs& A, cudaStream_t st);   // solve_pair.cu

cudaError_t dp_solve_upload_tables(dp_plan* P) {
  std::vector<double> t, frag;
  cudaError_t e = cudaErrorInvalidValue;
  const int nz = P->p.nz;
#define X(NZ) if (nz == NZ) { host_tables<NZ>(t, frag); e = cudaMemcpyToSymbol(c_tab##NZ, t.data(), sizeof(double) * t.size()); if (e == cudaSuccess) e = set_attr_nz<NZ>(); }
  DP_SOLVE_NZ_LIST(X)
#undef X
  if (e != cudaSuccess) return e;
  if (!P->d_solve_frag) {
    e = cudaMalloc(&P->d_solve_frag, sizeof(double) * frag.size());
    if (e != cudaSuccess) return e;
    P->device_bytes += sizeof(double) * frag.size();
    e = cudaMemcpy(P->d_solve_frag, frag.data(), sizeof(double) * frag.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
  }
  if (!P->d_ct_full) {
    typedef long double ld;
    const ld PI = 3.141592653589793238462643383279502884L;
    std::vector<double> ct((size_t)nz * nz);
    for (int n = 0; n < nz; ++n) for (int l = 0; l < nz; ++l) ct[(size_t)n * nz + l] = (double)cosl(PI * n * l / (nz - 1));
    e = cudaMalloc(&P->d_ct_full, sizeof(double) * ct.size());
    if (e != cudaSuccess) return e;
    P->device_bytes += sizeof(double) * ct.size();
    e = cudaMemcpy(P->d_ct_full, ct.data(), sizeof(double) * ct.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
  }
  if (!P->solve_pair_tab && dp_solve_pair_supports_nz(nz)) e = dp_solve_pair_create(P);
  return e;
}

void dp_solve_destroy_tables(dp_plan* P) {
  if (P->d_ct_full) { cudaFree(P->d_ct_full); P->d_ct_full = nullptr; }
  if (P->d_solve_frag) { cudaFree(P->d_solve_frag); P->d_solve_frag = nullptr; }
  dp_solve_pair_destroy(P);
}

cudaError_t dp_launch_solve(dp_plan* P, bool with_torque_field, bool want_omega, cudaStream_t st) {
  SolveArgs A;
  A.cplx = P->d_cplx; A.cplx_field = P->cplx_field;
  A.nx = P->p.nx; A.ny = P->p.ny; A.nkx = P->nkx;
  A.n_fast = P->nkx; A.n_slow = P->p.ny; A.pitch = P->nkxp; A.fast_is_x = 1; A.ky_of_pos = nullptr; A.lmin = P->d_lmin;
  if (P->own_fft) { A.n_fast = P->p.ny; A.n_slow = P->nkx; A.pitch = P->p.ny; A.fast_is_x = 0; A.ky_of_pos = dp_fft_own_ky_table(P); }
  A.frag = P->d_solve_frag;
  A.Lx = P->p.Lx; A.Ly = P->p.Ly; A.H = P->p.H; A.eta = P->p.eta;
  A.wall_mode = P->p.wall_mode; A.torque = with_torque_field ? 1 : 0; A.omega = want_omega ? 1 : 0;
  A.l0 = P->p.slip_0; A.lH = P->p.slip_H;
  A.slip = (P->p.wall_mode == DP_SLIT && (A.l0 != 0.0 || A.lH != 0.0)) ? 1 : 0;
  for (int c = 0; c < 2; ++c) { A.uw0[c] = P->p.uwall_0[c]; A.uwH[c] = P->p.uwall_H[c]; }
  cudaError_t e = cudaErrorInvalidValue;
  // three fields each way (no torque field to curl, no Omega field): the register-resident warp-pair kernel (solve_pair.cu);
  // dp_params.solve_kernel = 1 keeps this file's tile kernel (comparison runs)
  if (!A.torque && !A.omega && P->solve_pair_tab && !P->solve_force_tile) {
    e = dp_launch_solve_pair(P, A, st);
  } else {
#define X(NZ) if (P->p.nz == NZ) e = launch_nz<NZ>(A, st);
    DP_SOLVE_NZ_LIST(X)
#undef X
  }
  if (e != cudaSuccess) return e;
  k_zero_mode<<<1, 64, 0, st>>>(A, P->p.nz, P->d_ct_full);
  return cudaGetLastError();
}
