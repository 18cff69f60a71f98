// solve_pair.cu — per-wavenumber kernel of the doubly-periodic Stokes solver for products with THREE grid fields each way
// (forces only, or torques through the derivative of the ES kernel): paper steps 2(z)-6, PAPER.md:326-331 —
//   Chebyshev analysis in z, pressure BVP (eqs 15, 17), velocity BVPs (eqs 18, 22, 24), wall correction (eqs 42-44 for one wall;
//   App. A (A5), (A6), (A8), (A10) for the slit), Chebyshev synthesis.  Same discrete problem as solve.cu: tau rows
//   0..nz-3 of (D^2 - k^2) y = r plus the two Dirichlet-to-Neumann rows, solved in Greengard's integration form as two parity-decoupled
//   tridiagonal chains with one border unknown each.
//
// B200 mapping: the fp64 pipe bounds this kernel (8.3 k algorithmic FMAs per mode against 18.8 GB of traffic at cfg 5), so everything
// is arranged for it to issue fp64 instructions and little else:
//  * a warp PAIR owns 16 consecutive modes of one spectrum row; a lane is (mode, re/im); warp 0 of the pair owns the EVEN Chebyshev
//    coefficients of every column, warp 1 the ODD ones.  With the fold cos(n (N-l) pi/N) = (-1)^n cos(n l pi/N) the transforms, the
//    chain factorisation and the four BVPs split exactly along that line, so each warp keeps its half of f_x, f_y, f_z (then p, then
//    u, v, w) in REGISTERS from the analysis to the synthesis;
//  * the transforms are 16 x 16 (nz = 32) matrix-vector products per lane whose matrix entries are the same for all lanes of a warp:
//    the tables travel as a __grid_constant__ kernel parameter and are read into uniform registers (LDCU; sm_100a has no constant-bank
//    operand on DFMA), each entry feeding the DFMAs of all three fields; the loops over the input (analysis) and output (synthesis)
//    index are ROLLED (unrolled by two): ~150 instructions that stay in the L0 instruction cache;
//  * the two parities meet in five places only — d/dz of f_z for the pressure right-hand side, d/dz of p for the w right-hand side, the
//    end-point sums (p(0), p(H), u_DP on the walls), and the un-fold g_l = E_l + O_l, g_{N-l} = E_l - O_l after the synthesis — each a
//    few rows handed over through shared memory behind a barrier;
//  * the nodal columns come in by cp.async (16 bytes per (mode, re/im) pair) while the warps factor their chains; the correction is
//    added at the nodes (analysis and synthesis are exact inverses of one another, so this equals adding its coefficients);
//  * one CTA = six pairs (12 warps, one CTA per SM at nz = 32) that step through the phases behind CTA-wide barriers: the chain sweeps
//    are ~3 k straight-line instructions per warp, executed once per 16 modes, and an SM cannot fetch that much code for warps that
//    are at different places in it (profiles/r2_b_fetch_microbenchmarks.md) — in step, the six warps of a parity share one fetch
//    stream; reciprocals and exponentials are branch-free for the same reason (no BSSY / BSYNC around library slow paths).
#include <cmath>
#include <cstring>
#include <vector>

#include "solve_common.cuh"

using namespace dp_solve;

namespace {

// geometry of a compiled nz: NE even coefficients / node pairs (l, N-l) incl. the middle node of an odd nz, NO odd coefficients
template <int NZ> struct PG {
  static constexpr int N = NZ - 1, NE = N / 2 + 1, NO = NZ - NE;
  static_assert(NE == (NZ + 1) / 2, "even coefficients = node pairs");
};

// tables of one plan: analysis A[par][l][j] (times 1/(nx ny): the inverse FFT is unnormalised; j = output index runs fastest, so the
// sixteen entries an input value meets are adjacent in the constant bank), synthesis S[par][l][j] (the coefficient index j fastest: an output value is a dot product with one row), boundary-row functionals
// P_n, Q_n (see chains()), nodes xi_l = cos(l pi/N)
template <int NZ> struct alignas(16) PairTab {
  static constexpr int NEP = (PG<NZ>::NE + 1) & ~1;      // rows padded to whole 16-byte pairs (LDCU.128)
  double A[2][PG<NZ>::NE][NEP];
  double S[2][PG<NZ>::NE][NEP];
  double P[NZ], Q[NZ], XI[NZ];
  // per-row constants of the chains (n = row index): rows d_n = 1 + kappa^2 RD[n], l_n = kappa^2 RL[n], u_n = kappa^2 RU[n] (0 beyond the last
  // row), and 1/(2n) for the integrations — one LDCU each instead of a pair of immediate moves
  double RD[NZ], RL[NZ], RU[NZ], IH[NZ + 1];
  double EC[12];                                        // 1/13! ... 1/2!: Taylor coefficients of dp_exp_neg's polynomial
};
struct PairConst { double s, inv_s, sc, inv_2eta, dkx, dky; };   // H/2, 2/H, (H/2)^2 / eta, 1/(2 eta), 2 pi / Lx, 2 pi / Ly: computed once on the host
template <int NZ> struct PairArgs {
  SolveArgs a;
  PairConst c;
  PairTab<NZ> t;
};

template <int NZ> struct PairSmem {
  static constexpr int ROW = LN;                          // doubles per row: one value per lane
  static constexpr int NB = 0;                            // [3][NZ][32] nodal columns; later the hand-over rows (see the kernel)
  static constexpr int FAC = NB + 3 * NZ * ROW;           // [2][NZ][TM] inverse pivots, border solution (by row n); later e^{-k z}
  static constexpr int IBG = FAC + 2 * NZ * TM;           // [2][TM] 1 / B_g of the even / odd chain
  static constexpr int GPQ = IBG + 2 * TM;                // [2][2][TM] sums of b_m and of c_n of the unit border solution (even / odd chain)
  static constexpr int SUM = GPQ + 4 * TM;                // [2][8][32] sums handed over: S_c of p, u, v, w and S_b of u, v per parity
  static constexpr int DOUBLES = SUM + 2 * 8 * ROW;
  // pairs per CTA and CTAs per SM: one CTA of six pairs (measured: two CTAs of three pairs 12.6 ms, three of two 11.9 ms, one of six
  // 10.9 ms at cfg 5 — the warps of one parity must run the SAME stretch of straight-line code at the same time, see the header)
  static constexpr int PAIRS_SM = (227 * 1024 - 2048) / (DOUBLES * 8);       // pairs whose shared memory fits one SM
#define DP_PAIR_CTAS 1
#define DP_PAIR_NPAIR 6
  static constexpr int CTAS = PAIRS_SM >= DP_PAIR_CTAS ? DP_PAIR_CTAS : 1;
  static constexpr int NPAIR = PAIRS_SM / CTAS >= DP_PAIR_NPAIR ? DP_PAIR_NPAIR : (PAIRS_SM / CTAS >= 1 ? PAIRS_SM / CTAS : 1);
  static constexpr int THREADS = 64 * NPAIR;
};

template <int NZ> __device__ __forceinline__ void pair_sync() { named_sync(0, PairSmem<NZ>::THREADS); }
// Ends a basic block without doing anything (the branch is never taken and costs one uniform compare): ptxas schedules block by
// block, so work of a later step cannot be started (and its operands loaded) long before its turn at the price of spills.
// The condition cannot hold: dp_create accepts only nx >= DP_TILE_X + w > 0 and the kernel is launched from a validated plan only.
// Bodies without a fatal effect were measured in round 3 and dropped: "nanosleep" 158 -> 162 registers and 10.64 -> 10.81 ms at cfg 5;
// "exit" / "brkpt" compile to 162 registers as well (nz = 40: 128 / 384 bytes of spill loads instead of 88).
#define DP_SPLIT(A, id) do { if ((A).nx == -(id)) asm volatile("trap;"); } while (0)
// keeps ptxas from hoisting the shared-memory loads of a later block of work above this point (register pressure)
__device__ __forceinline__ void sched_fence() { __syncwarp(); }

// ---- factorisation of the chain of parity PAR for this lane's mode (depends on |k| only): inverse pivots Fi[n], the solution Fa[n]
// with unit border unknown, and 1/B_g (B_g = boundary functional of that solution).  Rows are indexed by n with stride TM.
template <int NZ, int PAR>
__device__ __forceinline__ double factor_chain(const PairTab<NZ>& T, double* Fi, double* Fa, double* Gpq, double k, double k2,
                                               double inv_s, bool store) {
  constexpr int n0 = Ch<NZ, PAR>::n0, NR = Ch<NZ, PAR>::NR;
  double invd[NR], ag[NR];
  double g = PAR ? k2 : 0.25 * k2 * k2;
#pragma unroll
  for (int j = 0; j < NR; ++j) {
    const int n = n0 + 2 * j;
    double d = fma(k2, T.RD[n], 1.0);
    if (j > 0) {
      const double mu = k2 * T.RL[n] * invd[j - 1];
      d = fma(-mu, k2 * T.RU[n - 2], d);
      g = -mu * g;
    }
    invd[j] = dp_rcp(d);
    ag[j] = g;
  }
  double SP = 0.0, SQ = 0.0, next = 0.0;
#pragma unroll
  for (int j = NR - 1; j >= 0; --j) {
    const int n = n0 + 2 * j;
    const double a = (ag[j] - k2 * T.RU[n] * next) * invd[j];
    next = a;
    if (store) { Fa[n * TM] = a; Fi[n * TM] = invd[j]; }
    SP = fma(T.P[n], a, SP); SQ = fma(T.Q[n], a, SQ);
  }
  // sums of the first-integral coefficients b_m and of the coefficients c_n of this unit-border solution: a_0 = kappa^2 c_0 and c_0 = 1
  // itself (even chain); b_0 = 1, which is also c_1's leading term (odd chain)
  if (!PAR) { SP = fma(T.P[0], k2, SP); SQ = fma(T.Q[0], k2, SQ); }
  const double GP = PAR ? 1.0 + SP : SP, GQ = 1.0 + SQ;
  if (store) { Gpq[0] = GP; Gpq[TM] = GQ; }
  return dp_rcp(inv_s * GP + k * GQ);
}

// ---- NC BVPs at once on the chain of parity PAR of this lane (the factors are loaded once): forward elimination, back substitution
// with the boundary functional, border unknown, double integration.
//   in : a[c][j] = (H/2)^2 r_n of row n = n0 + 2j, rho0[c] = (H/2)^2 r_0 (even chain), beta_bc[c] = this chain's boundary datum
//   out: cc[c][i] = coefficient c_n of y, n = PAR + 2i (i < NH);  bo[c][i] = first-integral coefficient b_{n+1} = (H/2)(dy/dz)_{n+1},
//        n = PAR + 2i — they carry the OTHER parity; border[c] = c_0 (even chain) or b_0 (odd chain);  Sc[c] = sum of the c_n;
//        Sb[c] = sum of the b_m this chain produces (wall derivatives for partial slip, footnote 46)
template <int NZ, int PAR, int NC>
__device__ __forceinline__ void chains(const SolveArgs& A, const PairTab<NZ>& T, double (&a)[NC][Ch<NZ, PAR>::NR], const double (&rho0)[NC], const double (&beta_bc)[NC],
                                       const double* Fi, const double* Fa, const double* Gpq, double k, double k2, double inv_s, double invBg,
                                       double (&cc)[NC][PAR ? PG<NZ>::NO : PG<NZ>::NE], double (&bo)[NC][PAR ? PG<NZ>::NO : PG<NZ>::NE],
                                       double (&border)[NC], double (&Sc)[NC], double (&Sb)[NC]) {
  constexpr int N = NZ - 1, n0 = Ch<NZ, PAR>::n0, NR = Ch<NZ, PAR>::NR;
  if (!PAR) {
#pragma unroll
    for (int c = 0; c < NC; ++c) a[c][0] = fma(0.25 * k2, rho0[c], a[c][0]);     // even chain: row 2 carries (kappa^2/4) rho_0
  }
#pragma unroll
  for (int j = 1; j < NR; ++j) {
    const double mu = k2 * T.RL[n0 + 2 * j] * Fi[(n0 + 2 * j - 2) * TM];
#pragma unroll
    for (int c = 0; c < NC; ++c) a[c][j] = fma(-mu, a[c][j - 1], a[c][j]);
  }
  DP_SPLIT(A, 1);
  double SP[NC], SQ[NC], next[NC];
#pragma unroll
  for (int c = 0; c < NC; ++c) SP[c] = SQ[c] = next[c] = 0.0;
#pragma unroll
  for (int j = NR - 1; j >= 0; --j) {
    const int n = n0 + 2 * j;
    const double ru = k2 * T.RU[n], fi = Fi[n * TM];
#pragma unroll
    for (int c = 0; c < NC; ++c) {
      const double v = fma(-ru, next[c], a[c][j]) * fi;
      a[c][j] = v; next[c] = v;
      SP[c] = fma(T.P[n], v, SP[c]); SQ[c] = fma(T.Q[n], v, SQ[c]);
    }
  }
  // border unknown from the boundary row; the sums of the b_m and of the c_n of the solution follow from the same functionals
  // (S_b = SP + border G_P, S_c = SQ + border G_Q with the unit border solution's sums G_P, G_Q): no summation of the results
  const double GP = Gpq[0], GQ = Gpq[TM];
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    if (!PAR) { SP[c] = fma(T.P[0], rho0[c], SP[c]); SQ[c] = fma(T.Q[0], rho0[c], SQ[c]); }
    border[c] = (beta_bc[c] - (inv_s * SP[c] + k * SQ[c])) * invBg;               // c_0 (even chain) or b_0 (odd chain)
    Sb[c] = fma(border[c], GP, SP[c]);
    Sc[c] = fma(border[c], GQ, SQ[c]);
  }
  DP_SPLIT(A, 2);
#pragma unroll
  for (int j = 0; j < NR; ++j) {
    const double fa = Fa[(n0 + 2 * j) * TM];
#pragma unroll
    for (int c = 0; c < NC; ++c) a[c][j] = fma(border[c], fa, a[c][j]);
  }
  // integrate twice:  b_{n+1} = (cbar_n a_n - a_{n+2}) / (2(n+1)),  c_n = (cbar_{n-1} b_{n-1} - b_{n+1}) / (2n)
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    DP_SPLIT(A, 3 + c);
    double bprev;
    if (!PAR) { cc[c][0] = border[c]; bprev = 0.0; }
    else bprev = border[c];
#pragma unroll
    for (int i = 0; i <= (N - PAR) / 2; ++i) {
      const int n = PAR + 2 * i;
      // a_n of parity PAR: n = 0 -> rho0 + border kappa^2 (even); n = n0 + 2j -> a[j]; n > N-2 -> 0
      double an = 0.0, ap = 0.0;
      if (n <= N - 2) an = (!PAR && n == 0) ? fma(border[c], k2, rho0[c]) : a[c][n >= n0 ? (n - n0) / 2 : 0];
      if (n + 2 <= N - 2) ap = a[c][(n + 2 - n0) / 2];
      const double bn1 = ((n == 0 ? 2.0 : 1.0) * an - ap) * T.IH[n + 1];
      if (n >= 1) cc[c][i] = ((n == 1 ? 2.0 : 1.0) * bprev - bn1) * T.IH[n];
      bo[c][i] = (n + 1 <= N - 1) ? bn1 : 0.0;
      bprev = bn1;
    }
  }
}

// ---- last step for the warp of parity PAR: its own nodes (l for the even warp, N - l for the odd one) from E_l, O_l in the
// buffer, plus the correction evaluated at the node, to global memory
template <int NZ, int PAR, bool SLIT>
__device__ __forceinline__ void store_nodes(const PairTab<NZ>& T, const double* NB, const double* EXP, const double (&cf)[3][4], double* gout,
                                            size_t cplx_field, size_t plane, double s, int lane, bool store_ok, int lm) {
  typedef PG<NZ> G;
  constexpr int N = G::N, NE = G::NE, NO = G::NO, NH = PAR ? NO : NE, VS = NZ * LN;
  const int mode = lane >> 1;
  // own nodes that are stored: l >= lm for the even warp, N - l >= lm for the odd one
  const int lmc = lm < 0 ? 0 : lm;
  const int lbeg = PAR ? 0 : (lmc < NH ? lmc : NH), lend = PAR ? ((N - lmc + 1) < NH ? (N - lmc + 1 > 0 ? N - lmc + 1 : 0) : NH) : NH;
#pragma unroll 2
  for (int l = lbeg; l < lend; ++l) {
    const int node = PAR ? N - l : l;
    const bool mid = (!PAR && l >= NO);                  // the middle node of an odd nz: no O row, and it mirrors itself
    const double z = s * (1.0 + T.XI[node]);
    const double e1 = EXP[(PAR * NE + l) * TM + mode];
    // e^{-k(H-z)} = the partner's e^{-kz} at the mirrored node
    const double e2 = SLIT ? (mid ? e1 : EXP[((1 - PAR) * NE + (mid ? 0 : l)) * TM + mode]) : 0.0;
    double* go = gout + 2 * (size_t)node * plane;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double ve = NB[c * VS + l * LN + lane];
      const double vo = mid ? 0.0 : NB[c * VS + (NE + (mid ? 0 : l)) * LN + lane];
      double v = PAR ? ve - vo : ve + vo;
      v = fma(fma(cf[c][0], z, cf[c][1]), e1, v);
      if (SLIT) v = fma(fma(cf[c][2], z, cf[c][3]), e2, v);
      if (store_ok && node >= lm) go[2 * (size_t)c * cplx_field] = v;       // planes above every footprint are never interpolated from
    }
  }
}

// ptxas schedules the whole unrolled body as one block and would start later phases (exponentials, boundary data) early at the
// price of spills: every phase therefore re-reads the mode constants from shared memory BEHIND its barrier
__device__ __forceinline__ ModeK load_modek(const double* SUM, int lane) {
  ModeK K;
  K.k = SUM[6 * LN + lane]; K.k2 = SUM[7 * LN + lane]; K.kxt = SUM[14 * LN + lane]; K.kyt = SUM[15 * LN + lane];
  K.sgI = (lane & 1) ? 1.0 : -1.0;
  return K;
}

template <int NZ, int PAR>
__device__ __forceinline__ void pair_body(const PairArgs<NZ>& PA, double* smem, const int lane, const bool store_ok,
                                          const size_t plane, const size_t off0) {
  typedef PG<NZ> G;
  typedef PairSmem<NZ> S;
  constexpr int N = G::N, NE = G::NE, NO = G::NO, NH = PAR ? NO : NE, NR = Ch<NZ, PAR>::NR, n0 = Ch<NZ, PAR>::n0;
  constexpr int VS = NZ * LN;
  const SolveArgs& A = PA.a;
  const PairTab<NZ>& T = PA.t;
  const int mode = lane >> 1, part = lane & 1;
  const double s = PA.c.s, inv_s = PA.c.inv_s;
  double* NB = smem + S::NB;
  const double* Fi = smem + S::FAC + mode;
  const double* Fa = smem + S::FAC + NZ * TM + mode;
  const double* Gpq = smem + S::GPQ + PAR * 2 * TM + mode;
  double* SUM = smem + S::SUM;
  const double invBg = smem[S::IBG + PAR * TM + mode];

  // ---- 1. Chebyshev analysis of the folded nodal columns (step 2): f^[c][j] = sum_l A[PAR][j][l] (g_l +- g_{N-l})
  // (the three fields go together: an entry of the table, fetched once from the constant bank, feeds three DFMAs)
  double f[3][NH];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int j = 0; j < NH; ++j) f[c][j] = 0.0;
  // a rolled loop over the input index l (the accumulators f are indexed statically): ~75 instructions that stay in the L0
  // instruction cache instead of 1500 fetched once
#pragma unroll 2
  for (int l = 0; l < NH; ++l) {
    double x[3];
    const bool alone = (N - l == l);                     // the middle node of an odd nz
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double ga = NB[c * VS + l * LN + lane];
      const double gb = alone ? 0.0 : NB[c * VS + (N - l) * LN + lane];
      x[c] = PAR ? ga - gb : ga + gb;
    }
    const double2* t = reinterpret_cast<const double2*>(&T.A[PAR][l][0]);
#pragma unroll
    for (int j = 0; j < NH; j += 2) {
      const double2 tt = t[j >> 1];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        f[c][j] = fma(tt.x, x[c], f[c][j]);
        if (j + 1 < NH) f[c][j + 1] = fma(tt.y, x[c], f[c][j + 1]);
      }
    }
  }
  pair_sync<NZ>();                                   // both warps have read the nodal columns: the buffer now carries the hand-overs

  // hand-over rows inside the old nodal buffer (each [32] doubles); X1, X2: NZ rows each; X4 = the whole buffer (written after the
  // last read of X1, X2: barrier 4 lies between)
  double* X1 = NB;                               // rows [0, nz): suffix sums of 2 m f^z_m, by index of the writer (even warp first)
  double* X2 = NB + NZ * LN;                     // rows [nz, 2 nz): (H/2) dp/dz coefficients, by index of the READER (odd reader first)
  double* ST = NB + (2 * NZ + PAR * NE) * LN;    // rows [2 nz, 3 nz): f^y waits here while the pressure is solved (registers)
#pragma unroll
  for (int j = 0; j < NH; ++j) ST[j * LN + lane] = f[1][j];

  // ---- 2. d/dz f^z couples the parities: (D g)_n = (2/H) sum_{m > n, m - n odd} 2 m g_m (n = 0 halved); hand the suffix sums over
  {
    double d = 0.0;
#pragma unroll
    for (int j = NH - 1; j >= 0; --j) {
      const int m = 2 * j + PAR;
      d = fma(2.0 * m, f[2][j], d);
      X1[(PAR * NE + j) * LN + lane] = d;
    }
  }
  pair_sync<NZ>();

  // ---- 3. pressure BVP (eqs 15, 17): r = i k.f + dz f_z;  i z: own part = sgI * other part
  double pc[1][NH];
  {
    const ModeK K = load_modek(SUM, lane);
    double a[1][NR], rho0[1] = {0.0}, bbc[1] = {0.0};
    const double s2 = s * s;
#pragma unroll
    for (int j = 0; j < NH; ++j) {
      const int n = 2 * j + PAR;
      if (n <= N - 2) {
        const double q = fma(K.kxt, f[0][j], K.kyt * ST[j * LN + lane]);
        const double qo = __shfl_xor_sync(0xffffffffu, q, 1);
        const int jm = PAR ? j + 1 : j;          // index of coefficient m = n + 1 in the other parity's numbering
        const double d = (jm < (PAR ? NE : NO)) ? X1[((1 - PAR) * NE + jm) * LN + lane] : 0.0;
        const double r = fma(K.sgI, qo, d * (n == 0 ? 0.5 * inv_s : inv_s)) * s2;
        if (n >= n0) a[0][(n - n0) / 2] = r; else rho0[0] = r;
      }
    }
    double bo[1][NH], border[1], Sc[1], Sb[1];
    chains<NZ, PAR, 1>(A, T, a, rho0, bbc, Fi, Fa, Gpq, K.k, K.k2, inv_s, invBg, pc, bo, border, Sc, Sb);
    // (H/2) dp/dz: the even chain yields b_m for odd m = 2i + 1 (reader index i), the odd chain b_0 = border and b_m for even m = 2i + 2
    if (!PAR) {
#pragma unroll
      for (int i = 0; i < NO; ++i) X2[i * LN + lane] = (i < NH) ? bo[0][i] : 0.0;
    } else {
      X2[(NO + 0) * LN + lane] = border[0];
#pragma unroll
      for (int i = 0; i + 1 < NE; ++i) X2[(NO + i + 1) * LN + lane] = (i < NH) ? bo[0][i] : 0.0;
    }
    SUM[(PAR * 8 + 0) * LN + lane] = Sc[0];
  }
  pair_sync<NZ>();

  // ---- 4. velocity BVPs (eq 18) with BCs (22), (24), the three components together (one load of the factors, three independent
  // dependency chains per lane)
  double uc[3][NH];
  {
    const ModeK K = load_modek(SUM, lane);
    const double se = SUM[(0 * 8 + 0) * LN + lane], so = SUM[(1 * 8 + 0) * LN + lane];
    const double pH = se + so, p0 = se - so;               // p(H) = sum p_n, p(0) = sum (-1)^n p_n ("direct summation")
    const double pHo = __shfl_xor_sync(0xffffffffu, pH, 1), p0o = __shfl_xor_sync(0xffffffffu, p0, 1);
    const double sc = PA.c.sc, inv_2eta = PA.c.inv_2eta;
    double a[3][NR], rho0[3] = {0.0, 0.0, 0.0}, bbc[3];
    const double fu = K.sgI * K.kxt, fv = K.sgI * K.kyt;
#pragma unroll
    for (int j = 0; j < NH; ++j) {
      const int n = 2 * j + PAR;
      if (n <= N - 2) {
        // r = (i k_c p - f_c)/eta (c = x, y);  r = (dz p - f_z)/eta
        const double po = __shfl_xor_sync(0xffffffffu, pc[0][j], 1);
        const double dzp = X2[((PAR ? 0 : NO) + j) * LN + lane] * inv_s;
        const double ru = fma(fu, po, -f[0][j]) * sc, rv = fma(fv, po, -ST[j * LN + lane]) * sc, rw = (dzp - f[2][j]) * sc;
        if (n >= n0) { a[0][(n - n0) / 2] = ru; a[1][(n - n0) / 2] = rv; a[2][(n - n0) / 2] = rw; }
        else { rho0[0] = ru; rho0[1] = rv; rho0[2] = rw; }
      }
    }
    // (dz + k) u(H) = -(i k_c/(2 k eta)) p(H), (dz - k) u(0) = +(i k_c/(2 k eta)) p(0) (eq 22); (dz +- k) w = p/(2 eta) at z = H, 0 (eq 24)
    const double inv_k = dp_rcp(K.k);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double gH, g0;
      if (c < 2) {
        const double cfc = (c == 0 ? K.kxt : K.kyt) * inv_k * inv_2eta;
        gH = -K.sgI * cfc * pHo; g0 = K.sgI * cfc * p0o;
      } else {
        gH = pH * inv_2eta; g0 = p0 * inv_2eta;
      }
      bbc[c] = PAR ? 0.5 * (gH + g0) : 0.5 * (gH - g0);
    }
    double bo[3][NH], border[3], Sc[3], Sb[3];
    chains<NZ, PAR, 3>(A, T, a, rho0, bbc, Fi, Fa, Gpq, K.k, K.k2, inv_s, invBg, uc, bo, border, Sc, Sb);
#pragma unroll
    for (int c = 0; c < 3; ++c) SUM[(PAR * 8 + 1 + c) * LN + lane] = Sc[c];
    if (A.slip) { SUM[(PAR * 8 + 4) * LN + lane] = Sb[0]; SUM[(PAR * 8 + 5) * LN + lane] = Sb[1]; }
  }
  DP_SPLIT(A, 8);

  pair_sync<NZ>();                                   // barrier 4: the sums of both parities are in place; X1, X2, the parked f^y are dead
  // ---- 5. synthesis (step 7 in z): E_l = sum_j u^_{2j} cos(2j l pi/N) | O_l = sum_j u^_{2j+1} cos((2j+1) l pi/N), three fields together,
  // in two halves of l (registers); the results go to the old nodal buffer: row l of field c, even warp rows [0, NE), odd warp [NE, nz)
  // rolled over the OUTPUT index l, two at a time (six independent sums); the coefficients stay in registers
  {
    constexpr int LE = NH & ~1;
#pragma unroll 2
    for (int l = 0; l < LE; l += 2) {
      const double2* t0 = reinterpret_cast<const double2*>(&T.S[PAR][l][0]);
      const double2* t1 = reinterpret_cast<const double2*>(&T.S[PAR][l + 1][0]);
      double g0[3] = {0.0, 0.0, 0.0}, g1[3] = {0.0, 0.0, 0.0};
#pragma unroll
      for (int j = 0; j < NH; j += 2) {
        const double2 ta = t0[j >> 1], tb = t1[j >> 1];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          g0[c] = fma(ta.x, uc[c][j], g0[c]); g1[c] = fma(tb.x, uc[c][j], g1[c]);
          if (j + 1 < NH) { g0[c] = fma(ta.y, uc[c][j + 1], g0[c]); g1[c] = fma(tb.y, uc[c][j + 1], g1[c]); }
        }
      }
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        NB[c * VS + ((PAR ? NE : 0) + l) * LN + lane] = g0[c];
        NB[c * VS + ((PAR ? NE : 0) + l + 1) * LN + lane] = g1[c];
      }
    }
    if (NH & 1) {
      const double* t0 = &T.S[PAR][NH - 1][0];
      double g0[3] = {0.0, 0.0, 0.0};
#pragma unroll
      for (int j = 0; j < NH; ++j)
#pragma unroll
        for (int c = 0; c < 3; ++c) g0[c] = fma(t0[j], uc[c][j], g0[c]);
#pragma unroll
      for (int c = 0; c < 3; ++c) NB[c * VS + ((PAR ? NE : 0) + NH - 1) * LN + lane] = g0[c];
    }
  }
  const ModeK K = load_modek(SUM, lane);
  // e^{-k z} at this warp's own nodes, z_l (even warp) or z_{N-l} = H - z_l (odd warp): the two parts of a mode share the work and
  // leave the values in shared memory (the chain factors are dead); the slit also needs those of the mirrored nodes = the partner's
  double* EXP = smem + S::FAC;
  const int lm = __ldg(A.lmin);                  // nodes l < lm are not stored (no footprint reaches them)
  {
    constexpr int HALF = (NH + 1) / 2;
#pragma unroll
    for (int i = 0; i < HALF; ++i) {             // unrolled: the exponentials are independent dependency chains
      const int l = 2 * i + part;
      if (l < NH) {
        const double xi = part ? T.XI[2 * i + 1 < NH ? 2 * i + 1 : 0] : T.XI[2 * i];
        const double z = s * (PAR ? 1.0 - xi : 1.0 + xi);
        EXP[(PAR * NE + l) * TM + mode] = dp_exp_neg_tab(-K.k * z, T.EC);
      }
    }
  }

  // ---- 6. wall correction coefficients (both warps, redundantly): u_DP on the walls by direct summation
  double cf[3][4];
  {
    double ssum[6], ssb[4];
#pragma unroll
    for (int c = 0; c < 3; ++c) { ssum[c * 2 + 0] = SUM[(0 * 8 + 1 + c) * LN + lane]; ssum[c * 2 + 1] = SUM[(1 * 8 + 1 + c) * LN + lane]; }
#pragma unroll
    for (int c = 0; c < 2; ++c) { ssb[c * 2 + 0] = A.slip ? SUM[(0 * 8 + 4 + c) * LN + lane] : 0.0; ssb[c * 2 + 1] = A.slip ? SUM[(1 * 8 + 4 + c) * LN + lane] : 0.0; }
    correction_coefficients(ssum, ssb, K, A.H, A.wall_mode, A.l0, A.lH, cf);
  }
  pair_sync<NZ>();                                   // barrier 5

  // ---- 7. back to the nodes g_l = E_l + O_l (even warp, l < NE), g_{N-l} = E_l - O_l (odd warp, l < NO); correction at the node
  // (basis z e^{-kz}, e^{-kz}, z e^{-k(H-z)}, e^{-k(H-z)}); store.  A rolled loop per geometry.
  double* gout = reinterpret_cast<double*>(A.cplx) + 2 * off0 + part;
  if (A.wall_mode == DP_SLIT) store_nodes<NZ, PAR, true>(T, NB, EXP, cf, gout, A.cplx_field, plane, s, lane, store_ok, lm);
  else store_nodes<NZ, PAR, false>(T, NB, EXP, cf, gout, A.cplx_field, plane, s, lane, store_ok, lm);
}

template <int NZ>
__global__ void __launch_bounds__(PairSmem<NZ>::THREADS, PairSmem<NZ>::CTAS) k_solve_pair(const __grid_constant__ PairArgs<NZ> PA) {
  extern __shared__ __align__(16) double smem_cta[];
  typedef PairSmem<NZ> S;
  const int pair = threadIdx.x >> 6;
  double* smem = smem_cta + pair * S::DOUBLES;
  constexpr int VS = NZ * LN;
  const SolveArgs& A = PA.a;
  const int tid = threadIdx.x & 63, lane = tid & 31, wid = tid >> 5;
  const int mode = lane >> 1, part = lane & 1;
  const int fast0 = (blockIdx.x * S::NPAIR + pair) * TM;
  const int ifast = fast0 + mode, islow = blockIdx.y;
  const bool valid = ifast < A.n_fast;
  const int ix = A.fast_is_x ? ifast : islow;
  const int iy = A.fast_is_x ? islow : ((A.ky_of_pos && valid) ? __ldg(A.ky_of_pos + ifast) : ifast);
  const bool zero_mode = (ix == 0 && iy == 0);
  const double s = PA.c.s, inv_s = PA.c.inv_s;
  ModeK K;
  K.k = 1.0; K.kxt = 0.0; K.kyt = 0.0; K.sgI = part ? 1.0 : -1.0;
  if (valid && !zero_mode) {
    const int nyq = (iy <= A.ny / 2) ? iy : iy - A.ny;
    const double kx = PA.c.dkx * ix, ky = PA.c.dky * nyq;
    K.k = sqrt(kx * kx + ky * ky);                         // magnitude: always the full values (reading G5)
    K.kxt = (ix == A.nx / 2) ? 0.0 : kx;                   // component multipliers vanish on the unpaired Nyquist index
    K.kyt = (iy == A.ny / 2) ? 0.0 : ky;
  }
  K.k2 = (K.k * s) * (K.k * s);
  const size_t plane = (size_t)A.n_slow * A.pitch;
  const size_t off0 = (size_t)islow * A.pitch + ifast;

  // ---- 0. nodal columns HBM -> shared memory, 16 bytes ((re, im) of one mode) per copy: a half warp moves one row (field, node)
  {
    const int lm = __ldg(A.lmin);
    const int sub = lane >> 4, m = lane & 15;
    const int mfast = fast0 + m;
    const bool mvalid = mfast < A.n_fast;
    const size_t moff = (size_t)islow * A.pitch + mfast;
    // half warp (wid, sub) takes the nodes l = 2 wid + sub, + 4, ... of every field: pointers advance by constant strides
    const int l0 = 2 * wid + sub;
    const double2* src = A.cplx + (size_t)l0 * plane + moff;
    double* dst = &smem[S::NB + l0 * LN + 2 * m];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double2* sp = src;
      double* dp = dst;
#pragma unroll 4
      for (int l = l0; l < NZ; l += 4) {
        if (mvalid && l >= lm) cp_async16(dp, sp);
        else *reinterpret_cast<double2*>(dp) = make_double2(0.0, 0.0);
        sp += 4 * plane; dp += 4 * LN;
      }
      src += A.cplx_field; dst += VS;
    }
    cp_async_commit();
  }
  // the chain of this warp's parity is factored in the shadow of the loads
  {
    double* Fi = smem + S::FAC + mode;
    double* Fa = smem + S::FAC + NZ * TM + mode;
    double ib;
    double* Gpq = smem + S::GPQ + wid * 2 * TM + mode;
    if (wid == 0) ib = factor_chain<NZ, 0>(PA.t, Fi, Fa, Gpq, K.k, K.k2, inv_s, part == 0);
    else ib = factor_chain<NZ, 1>(PA.t, Fi, Fa, Gpq, K.k, K.k2, inv_s, part == 0);
    if (part == 0) smem[S::IBG + wid * TM + mode] = ib;
    if (wid == 0) { smem[S::SUM + 6 * LN + lane] = K.k; smem[S::SUM + 7 * LN + lane] = K.k2; }
    else { smem[S::SUM + 14 * LN + lane] = K.kxt; smem[S::SUM + 15 * LN + lane] = K.kyt; }
  }
  cp_async_wait_all();
  pair_sync<NZ>();
  const bool store_ok = valid && !zero_mode;
  if (wid == 0) pair_body<NZ, 0>(PA, smem, lane, store_ok, plane, off0);
  else pair_body<NZ, 1>(PA, smem, lane, store_ok, plane, off0);
}

template <int NZ> void host_pair_tab(PairTab<NZ>& T, double scale) {
  typedef long double ld;
  typedef PG<NZ> G;
  const ld PI = 3.141592653589793238462643383279502884L;
  constexpr int N = NZ - 1;
  std::memset(&T, 0, sizeof(T));
  auto ctil = [&](int i) { return (i == 0 || i == N) ? (ld)2 : (ld)1; };
  for (int par = 0; par < 2; ++par) {
    const int nh = par ? G::NO : G::NE;
    for (int j = 0; j < nh; ++j)
      for (int l = 0; l < nh; ++l) {
        const int n = 2 * j + par;
        T.A[par][l][j] = (double)((ld)scale * (2 / (ld)N) / (ctil(n) * ctil(l)) * cosl(PI * (ld)n * l / N));
        T.S[par][l][j] = (double)cosl(PI * (ld)n * l / N);
      }
  }
  for (int l = 0; l <= N; ++l) T.XI[l] = (double)cosl(PI * l / N);
  for (int n = 1; n <= N; ++n) {             // the chain rows of solve_common.cuh's row_d / row_l / row_u, without the factor kappa^2
    T.RD[n] = n == 1 ? 0.125 : 1.0 / (2.0 * (n * n - 1));
    T.RL[n] = n >= 2 ? -(n == 2 ? 2.0 : 1.0) / (4.0 * n * (n - 1)) : 0.0;
    T.RU[n] = (n + 2 <= NZ - 3) ? -1.0 / (4.0 * n * (n + 1)) : 0.0;
  }
  for (int n = 1; n <= N + 1; ++n) T.IH[n] = 1.0 / (2.0 * n);
  { double f = 2.0; for (int q = 2; q <= 13; ++q) { T.EC[13 - q] = 1.0 / f; f *= (q + 1); } }   // EC[0] = 1/13!, ..., EC[11] = 1/2!
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
    T.P[n] = (double)p; T.Q[n] = (double)q;
  }
}

template <int NZ> size_t pair_smem_bytes() { return sizeof(double) * (size_t)PairSmem<NZ>::DOUBLES * PairSmem<NZ>::NPAIR; }

}  // namespace

// compiled sizes: the tables of larger nz do not fit a kernel parameter (32 KB); those plans keep the tile kernel of solve.cu
#define DP_PAIR_NZ_LIST(X) X(16) X(19) X(24) X(26) X(32) X(40) X(48)

bool dp_solve_pair_supports_nz(int nz) {
#define X(NZ) if (nz == NZ) return true;
  DP_PAIR_NZ_LIST(X)
#undef X
  return false;
}

cudaError_t dp_solve_pair_create(dp_plan* P) {
  const double scale = 1.0 / ((double)P->p.nx * (double)P->p.ny);
  cudaError_t e = cudaErrorInvalidValue;
#define X(NZ) if (P->p.nz == NZ) { PairTab<NZ>* t = new PairTab<NZ>; host_pair_tab<NZ>(*t, scale); P->solve_pair_tab = t; \
    e = cudaFuncSetAttribute(k_solve_pair<NZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pair_smem_bytes<NZ>()); }
  DP_PAIR_NZ_LIST(X)
#undef X
  return e;
}

void dp_solve_pair_destroy(dp_plan* P) {
  if (!P->solve_pair_tab) return;
#define X(NZ) if (P->p.nz == NZ) delete static_cast<PairTab<NZ>*>(P->solve_pair_tab);
  DP_PAIR_NZ_LIST(X)
#undef X
  P->solve_pair_tab = nullptr;
}

cudaError_t dp_launch_solve_pair(dp_plan* P, const SolveArgs& A, cudaStream_t st) {
  cudaError_t e = cudaErrorInvalidValue;
#define X(NZ) if (P->p.nz == NZ) { PairArgs<NZ> PA; PA.a = A; PA.c.s = 0.5 * A.H; PA.c.inv_s = 2.0 / A.H; PA.c.sc = 0.25 * A.H * A.H / A.eta; PA.c.inv_2eta = 0.5 / A.eta; PA.c.dkx = 2.0 * M_PI / A.Lx; PA.c.dky = 2.0 * M_PI / A.Ly; PA.t = *static_cast<const PairTab<NZ>*>(P->solve_pair_tab); \
    constexpr int CM = TM * PairSmem<NZ>::NPAIR; dim3 grid((A.n_fast + CM - 1) / CM, A.n_slow); \
    k_solve_pair<NZ><<<grid, PairSmem<NZ>::THREADS, pair_smem_bytes<NZ>(), st>>>(PA); e = cudaGetLastError(); }
  DP_PAIR_NZ_LIST(X)
#undef X
  return e;
}
