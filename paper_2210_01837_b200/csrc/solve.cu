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
// B200 mapping: one CTA = 32 consecutive kx of one ky row (a warp of modes).  All per-mode vectors live in shared
// memory as [vector][n][mode] (mode fastest: conflict-free, and the HBM rows are 512-byte coalesced).  Work is split
// into phases of independent items (vector x parity for the cosine transforms, part x chain for the sweeps);
// each warp takes an item, its 32 lanes are the 32 modes, so the transform matrices are warp-uniform and come
// straight from the constant bank as immediate operands of the DFMAs (fully unrolled, nz is a template parameter).
#include <cmath>
#include <vector>

#include "common.cuh"

namespace {

constexpr int TM = DP_SOLVE_TM;
constexpr int SOLVE_THREADS = 256;
constexpr int NWARPS = SOLVE_THREADS / 32;
constexpr int NVEC = 13;      // real shared-memory vectors per mode (see kernel)

// ---- constant tables per compiled nz: CT[n][l] = cos(n l pi/N) (n = 0..N, l < nz/2), P[n], Q[n] (boundary-row
//      functionals of a unit a_n, see kernel), XI[l] = cos(l pi/N)
template <int NZ> struct Tab {
  static constexpr int CT = 0, P = NZ * (NZ / 2), Q = P + NZ, XI = Q + NZ, SIZE = XI + NZ;
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
  int nx, ny, nkx, nkxp;
  double Lx, Ly, H, eta;
  int wall_mode, torque, omega;
};

// ---- tridiagonal rows of a chain (n >= 1): d_n a_n + l_n a_{n-2} + u_n a_{n+2}
template <int NZ> __device__ __forceinline__ double row_d(int n, double k2) { return n == 1 ? 1.0 + k2 * 0.125 : 1.0 + k2 / (2.0 * (n * n - 1)); }
template <int NZ> __device__ __forceinline__ double row_l(int n, double k2) { return -k2 * (n == 2 ? 2.0 : 1.0) / (4.0 * n * (n - 1)); }
template <int NZ> __device__ __forceinline__ double row_u(int n, double k2) { return (n + 2 <= NZ - 3) ? -k2 / (4.0 * n * (n + 1)) : 0.0; }

// ---- DCT-I analysis of one real vector, one output parity (items of phases 1 and 6b)
//   g^_n = (2/N)(1/c~_n) sum_l (1/c~_l) g_l cos(n l pi/N), folded with cos(n (N-l) pi/N) = (-1)^n cos(n l pi/N)
template <int NZ> __device__ __forceinline__ void analysis_load(const double* v, int par, double* e) {
  constexpr int N = NZ - 1, LH = NZ / 2;
#pragma unroll
  for (int l = 0; l < LH; ++l) {
    double a = v[l * TM], b = v[(N - l) * TM];
    e[l] = par ? a - b : a + b;
  }
  e[0] *= 0.5;
}
template <int NZ, int PAR> __device__ __forceinline__ void analysis_compute(double* v, const double* e) {
  constexpr int N = NZ - 1, LH = NZ / 2;
  const double* T = tab<NZ>();
#pragma unroll
  for (int j = 0; j < LH; ++j) {
    const int n = 2 * j + PAR;
    double acc = 0.0;
#pragma unroll
    for (int l = 0; l < LH; ++l) acc = fma(T[Tab<NZ>::CT + n * LH + l], e[l], acc);
    v[n * TM] = acc * ((n == 0 || n == N) ? 1.0 / N : 2.0 / N);
  }
}

// ---- DCT-I synthesis of one real vector: g_l = sum_n g^_n cos(n l pi/N)
template <int NZ> __device__ __forceinline__ void synthesis_inplace(double* v) {
  constexpr int N = NZ - 1, LH = NZ / 2;
  const double* T = tab<NZ>();
  double c[NZ];
#pragma unroll
  for (int n = 0; n < NZ; ++n) c[n] = v[n * TM];
#pragma unroll
  for (int l = 0; l < LH; ++l) {
    double E = 0.0, O = 0.0;
#pragma unroll
    for (int j = 0; j < LH; ++j) {
      E = fma(T[Tab<NZ>::CT + (2 * j) * LH + l], c[2 * j], E);
      O = fma(T[Tab<NZ>::CT + (2 * j + 1) * LH + l], c[2 * j + 1], O);
    }
    v[l * TM] = E + O;
    v[(N - l) * TM] = E - O;
  }
}

// ---- coefficient-space z-derivative, one output parity, top-down recurrence
//   d_N = 0, d_n = d_{n+2} + 2(n+1) g_{n+1},  (D g)_n = (2/H) d_n (d_0 halved)
//   dst[n] = scale * (D src)_n (+ dst[n] if ACC)
template <int NZ, bool ACC> __device__ __forceinline__ void deriv_sweep(const double* src, double* dst, int par, double inv_s, double scale) {
  constexpr int N = NZ - 1;
  double d = 0.0;
  const int ntop = ((N - par) & 1) ? N - 1 : N;       // largest n <= N with parity par
#pragma unroll
  for (int i = 0; i < NZ / 2; ++i) {
    const int n = ntop - 2 * i;
    if (n < 0) break;
    if (n + 1 <= N) d = fma(2.0 * (n + 1), src[(n + 1) * TM], d);
    const double val = d * inv_s * (n == 0 ? 0.5 : 1.0) * scale;
    if (ACC) dst[n * TM] += val; else dst[n * TM] = val;
  }
}

// ---- one chain of one BVP: forward elimination, back substitution with the boundary functional, border unknown,
//      double integration.  rho lives in col[n*TM] (own-parity slots, n <= N-2) and is overwritten by y's coefficients c_n.
//      If dcol != nullptr the first-integral coefficients b_n / s (= d y/dz) of the OTHER parity are stored there.
//      Returns S_c = sum of c_n over the chain (incl. c_0 for the even chain).
template <int NZ>
__device__ __forceinline__ double chain_solve(double* col, double* dcol, const double* mult, const double* invd, const double* ag,
                                              int par, double k, double k2, double inv_s, double beta_bc, double Bg) {
  constexpr int N = NZ - 1;
  const double* T = tab<NZ>();
  const int n0 = par ? 1 : 2;                    // first tridiagonal row
  const int nrows = par ? (N - 1) / 2 : (N - 2) / 2;   // rows n0, n0+2, ... <= N-2
  // forward elimination (rho'_j = rho_j - m_j rho'_{j-1}); even chain: row 2 carries (kappa^2/4) rho_0
  double prev = 0.0;
#pragma unroll
  for (int j = 0; j < NZ / 2; ++j) {
    const int n = n0 + 2 * j;
    if (j >= nrows) break;
    double r = col[n * TM];
    if (j == 0) { if (!par) r = fma(0.25 * k2, col[0], r); }
    else r = fma(-mult[n * TM], prev, r);
    col[n * TM] = r;
    prev = r;
  }
  // back substitution a_j = (rho'_j - u_j a_{j+1}) / d'_j, accumulating B = (1/s) sum P_n a_n + k sum Q_n a_n
  double SP = 0.0, SQ = 0.0, next = 0.0;
#pragma unroll
  for (int j = NZ / 2 - 1; j >= 0; --j) {
    const int n = n0 + 2 * j;
    if (j >= nrows) continue;
    double a = (col[n * TM] - row_u<NZ>(n, k2) * next) * invd[n * TM];
    col[n * TM] = a;
    next = a;
    SP = fma(T[Tab<NZ>::P + n], a, SP);
    SQ = fma(T[Tab<NZ>::Q + n], a, SQ);
  }
  if (!par) { const double a0 = col[0]; SP = fma(T[Tab<NZ>::P + 0], a0, SP); SQ = fma(T[Tab<NZ>::Q + 0], a0, SQ); }
  const double border = (beta_bc - (inv_s * SP + k * SQ)) / Bg;      // c_0 (even chain) or b_0 (odd chain)
  // integrate a = a^rho + border a^g twice:  b_{n+1} = (cbar_n a_n - a_{n+2}) / (2(n+1)),  c_n = (cbar_{n-1} b_{n-1} - b_{n+1}) / (2n)
  double Sc = 0.0, bprev;
  double an = fma(border, ag[par * TM], col[par * TM]);   // a_0 (even) or a_1 (odd)
  if (!par) { col[0] = border; Sc = border; bprev = 0.0; }
  else { if (dcol) dcol[0] = border * inv_s; bprev = border; }
#pragma unroll
  for (int i = 0; i < NZ / 2 + 1; ++i) {
    const int n = par + 2 * i;
    if (n > N) break;
    double ap = 0.0;
    if (n + 2 <= N - 2) ap = fma(border, ag[(n + 2) * TM], col[(n + 2) * TM]);
    const double bn1 = ((n == 0 ? 2.0 : 1.0) * an - ap) / (2.0 * (n + 1));
    if (n >= 1) {
      const double c = ((n == 1 ? 2.0 : 1.0) * bprev - bn1) / (2.0 * n);
      col[n * TM] = c;
      Sc += c;
    }
    if (dcol && n + 1 <= N - 1) dcol[(n + 1) * TM] = bn1 * inv_s;
    bprev = bn1;
    an = ap;
  }
  if (dcol) { if (((N - par) & 1) == 1) dcol[N * TM] = 0.0; }   // (D y)_N = 0: slot N belongs to the chain whose b's have N's parity
  return Sc;
}

// ---- 4x4 real system with two right-hand sides (real and imaginary part), partial pivoting after row equilibration
__device__ void solve4(double M[4][4], double br[4], double bi[4]) {
  for (int r = 0; r < 4; ++r) {
    double mx = fmax(fmax(fabs(M[r][0]), fabs(M[r][1])), fmax(fabs(M[r][2]), fabs(M[r][3])));
    double s = mx > 0.0 ? 1.0 / mx : 1.0;
    for (int c = 0; c < 4; ++c) M[r][c] *= s;
    br[r] *= s; bi[r] *= s;
  }
  for (int c = 0; c < 4; ++c) {
    int p = c; double best = fabs(M[c][c]);
    for (int r = c + 1; r < 4; ++r) if (fabs(M[r][c]) > best) { best = fabs(M[r][c]); p = r; }
    if (p != c) {
      for (int q = 0; q < 4; ++q) { double t = M[c][q]; M[c][q] = M[p][q]; M[p][q] = t; }
      double t = br[c]; br[c] = br[p]; br[p] = t; t = bi[c]; bi[c] = bi[p]; bi[p] = t;
    }
    for (int r = c + 1; r < 4; ++r) {
      double f = M[r][c] / M[c][c];
      for (int q = c; q < 4; ++q) M[r][q] -= f * M[c][q];
      br[r] -= f * br[c]; bi[r] -= f * bi[c];
    }
  }
  for (int r = 3; r >= 0; --r) {
    double sr = br[r], si = bi[r];
    for (int q = r + 1; q < 4; ++q) { sr -= M[r][q] * br[q]; si -= M[r][q] * bi[q]; }
    br[r] = sr / M[r][r]; bi[r] = si / M[r][r];
  }
}

template <int NZ>
__global__ void __launch_bounds__(SOLVE_THREADS, (NZ <= 32 ? 2 : 1)) k_solve(SolveArgs A) {
  extern __shared__ double smem[];
  constexpr int N = NZ - 1, LH = NZ / 2, VS = NZ * TM;
#define VEC(i) (smem + (size_t)(i) * VS)
  // vectors: 0..9 = five complex columns C0..C4 (re, im); 10 = Thomas multipliers, 11 = inverse pivots, 12 = a^g
  double* s_Bg = smem + (size_t)NVEC * VS;     // [2][TM]
  double* s_sum = s_Bg + 2 * TM;               // [4][2][2][TM]  S_c of (p,u,v,w) x (re,im) x (even,odd chain)
  double* s_corr = VEC(10);                    // [3][4][2][TM] correction coefficients (phases 6-7; factors are dead by then)
  const double* T = tab<NZ>();

  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int iy = blockIdx.y, ix = blockIdx.x * TM + lane;
  const bool valid = ix < A.nkx;
  const bool zero_mode = (ix == 0 && iy == 0);
  const double s = 0.5 * A.H, inv_s = 1.0 / s, eta = A.eta;
  double kx = 0.0, ky = 0.0, k = 1.0, kxt = 0.0, kyt = 0.0;
  if (valid && !zero_mode) {
    const int nyq = (iy <= A.ny / 2) ? iy : iy - A.ny;
    kx = 2.0 * M_PI * ix / A.Lx; ky = 2.0 * M_PI * nyq / A.Ly;
    k = sqrt(kx * kx + ky * ky);                           // magnitude: always the full values (reading G5)
    kxt = (ix == A.nx / 2) ? 0.0 : kx;                     // component multipliers vanish on the unpaired Nyquist index
    kyt = (iy == A.ny / 2) ? 0.0 : ky;
  }
  const double k2 = (k * s) * (k * s);
  const int m = lane;

  // ---------------- phase 0: load the nodal columns, fold the algebraic part of (1/2) curl t into f (eq 7)
  for (int l = wid; l < NZ; l += NWARPS) {
    double2 f[3] = {{0, 0}, {0, 0}, {0, 0}}, t[3] = {{0, 0}, {0, 0}, {0, 0}};
    if (valid) {
      const size_t off = ((size_t)l * A.ny + iy) * A.nkxp + ix;
#pragma unroll
      for (int c = 0; c < 3; ++c) f[c] = A.cplx[c * A.cplx_field + off];
      if (A.torque) {
#pragma unroll
        for (int c = 0; c < 3; ++c) t[c] = A.cplx[(3 + c) * A.cplx_field + off];
      }
    }
    const int o = l * TM + m;
    VEC(0)[o] = f[0].x - 0.5 * kyt * t[2].y;  VEC(1)[o] = f[0].y + 0.5 * kyt * t[2].x;
    VEC(2)[o] = f[1].x + 0.5 * kxt * t[2].y;  VEC(3)[o] = f[1].y - 0.5 * kxt * t[2].x;
    VEC(4)[o] = f[2].x - 0.5 * (kxt * t[1].y - kyt * t[0].y);
    VEC(5)[o] = f[2].y + 0.5 * (kxt * t[1].x - kyt * t[0].x);
    VEC(6)[o] = t[0].x; VEC(7)[o] = t[0].y; VEC(8)[o] = t[1].x; VEC(9)[o] = t[1].y;
  }
  __syncthreads();

  // ---------------- phase 1: Chebyshev analysis of the 3 (or 5) complex columns; item = (real vector, output parity)
  {
    const int items = (A.torque ? 10 : 6) * 2;
    for (int base = 0; base < items; base += NWARPS) {
      const int item = base + wid;
      const bool act = item < items;
      double e[LH];
      double* v = VEC(act ? item >> 1 : 0) + m;
      if (act) analysis_load<NZ>(v, item & 1, e);
      __syncthreads();
      if (act) { if (item & 1) analysis_compute<NZ, 1>(v, e); else analysis_compute<NZ, 0>(v, e); }
    }
  }
  __syncthreads();

  // ---------------- phase 2: chain factorisation + homogeneous solutions (2 items); D t_y, D t_x into f_x, f_y (8 items)
  {
    const int items = A.torque ? 10 : 2;
    for (int item = wid; item < items; item += NWARPS) {
      if (item < 2) {
        const int par = item;
        double* mult = VEC(10) + m; double* invd = VEC(11) + m; double* ag = VEC(12) + m;
        const int n0 = par ? 1 : 2, nrows = par ? (N - 1) / 2 : (N - 2) / 2;
        double dprev = 1.0, g = par ? k2 : 0.25 * k2 * k2;
#pragma unroll
        for (int j = 0; j < NZ / 2; ++j) {
          const int n = n0 + 2 * j;
          if (j >= nrows) break;
          double d = row_d<NZ>(n, k2);
          if (j > 0) {
            const double mu = row_l<NZ>(n, k2) / dprev;
            d = fma(-mu, row_u<NZ>(n - 2, k2), d);
            mult[n * TM] = mu;
            g = -mu * g;
          }
          invd[n * TM] = 1.0 / d;
          ag[n * TM] = g;
          dprev = d;
        }
        double SP = 0.0, SQ = 0.0, next = 0.0;
#pragma unroll
        for (int j = NZ / 2 - 1; j >= 0; --j) {
          const int n = n0 + 2 * j;
          if (j >= nrows) continue;
          const double a = (ag[n * TM] - row_u<NZ>(n, k2) * next) * invd[n * TM];
          ag[n * TM] = a; next = a;
          SP = fma(T[Tab<NZ>::P + n], a, SP); SQ = fma(T[Tab<NZ>::Q + n], a, SQ);
        }
        if (!par) {
          ag[0] = k2;                                      // a_0 = rho_0 + kappa^2 c_0
          SP = fma(T[Tab<NZ>::P + 0], k2, SP); SQ = fma(T[Tab<NZ>::Q + 0], k2, SQ);
          s_Bg[m] = inv_s * SP + k * (1.0 + SQ);           // c_0 = 1 also enters sum c_n directly
        } else {
          s_Bg[TM + m] = inv_s * (1.0 + SP) + k * (1.0 + SQ);   // b_0 = 1 enters sum b_n and c_1
        }
      } else {
        // f_x -= (1/2) D t_y ; f_y += (1/2) D t_x   (eq 7; the ik x t_z parts were folded in phase 0)
        const int q = item - 2, col = 3 + (q >> 2), part = (q >> 1) & 1, par = q & 1;
        const double* src = VEC(2 * col + part) + m;
        double* dst = (col == 4 ? VEC(0 + part) : VEC(2 + part)) + m;
        deriv_sweep<NZ, true>(src, dst, par, inv_s, col == 4 ? -0.5 : 0.5);
      }
    }
  }
  __syncthreads();

  // ---------------- phases 3+4: pressure right-hand side (eq 15) and pressure BVP with BCs (17); item = (part, chain)
  if (wid < 4) {
    const int part = wid >> 1, par = wid & 1;
    double* col = VEC(6 + part) + m;                      // C3 := p
    double* dcol = VEC(8 + part) + m;                     // C4 := dp/dz
    const double* fz = VEC(4 + part) + m;
    const double* fxo = VEC(0 + (1 - part)) + m;          // the OTHER part of f_x, f_y: i k f mixes re and im
    const double* fyo = VEC(2 + (1 - part)) + m;
    const double sg = part ? 1.0 : -1.0;                  // Re(i k f) = -k Im f ; Im(i k f) = +k Re f
    double d = 0.0;
    const int ntop = ((N - par) & 1) ? N - 1 : N;
#pragma unroll
    for (int i = 0; i < NZ / 2; ++i) {
      const int n = ntop - 2 * i;
      if (n < 0) break;
      if (n + 1 <= N) d = fma(2.0 * (n + 1), fz[(n + 1) * TM], d);
      double r = 0.0;
      if (n <= N - 2) r = sg * (kxt * fxo[n * TM] + kyt * fyo[n * TM]) + d * inv_s * (n == 0 ? 0.5 : 1.0);
      col[n * TM] = r * s * s;
    }
    const double Sc = chain_solve<NZ>(col, dcol, VEC(10) + m, VEC(11) + m, VEC(12) + m, par, k, k2, inv_s, 0.0, s_Bg[par * TM + m]);
    s_sum[((0 * 2 + part) * 2 + par) * TM + m] = Sc;
  }
  __syncthreads();

  // ---------------- phase 5: velocity BVPs (eq 18) with BCs (22), (24); item = (component, part, chain)
  for (int item = wid; item < 12; item += NWARPS) {
    const int comp = item >> 2, part = (item >> 1) & 1, par = item & 1;
    double* col = VEC(2 * comp + part) + m;               // f_c, overwritten by u_c
    const double pH_re = s_sum[(0 * 2 + 0) * 2 * TM + m] + s_sum[((0 * 2 + 0) * 2 + 1) * TM + m];
    const double p0_re = s_sum[(0 * 2 + 0) * 2 * TM + m] - s_sum[((0 * 2 + 0) * 2 + 1) * TM + m];
    const double pH_im = s_sum[(0 * 2 + 1) * 2 * TM + m] + s_sum[((0 * 2 + 1) * 2 + 1) * TM + m];
    const double p0_im = s_sum[(0 * 2 + 1) * 2 * TM + m] - s_sum[((0 * 2 + 1) * 2 + 1) * TM + m];
    double gH, g0;
    const int nlo = par ? 1 : 0;
    if (comp < 2) {
      const double kc = comp == 0 ? kxt : kyt;
      const double* po = VEC(6 + (1 - part)) + m;         // other part of p
      const double sg = part ? 1.0 : -1.0;
#pragma unroll
      for (int i = 0; i < NZ / 2; ++i) {
        const int n = nlo + 2 * i;
        if (n > N - 2) break;
        col[n * TM] = (sg * kc * po[n * TM] - col[n * TM]) * (s * s / eta);     // r = (i k_c p - f_c)/eta
      }
      const double c = kc / (2.0 * k * eta);
      // (dz + k) u(H) = -(i k_c/(2 k eta)) p(H) ; (dz - k) u(0) = +(i k_c/(2 k eta)) p(0)      (eq 22)
      gH = part ? -c * pH_re : c * pH_im;
      g0 = part ? c * p0_re : -c * p0_im;
    } else {
      const double* dp = VEC(8 + part) + m;
#pragma unroll
      for (int i = 0; i < NZ / 2; ++i) {
        const int n = nlo + 2 * i;
        if (n > N - 2) break;
        col[n * TM] = (dp[n * TM] - col[n * TM]) * (s * s / eta);              // r = (dz p - f_z)/eta
      }
      // (dz + k) w(H) = p(H)/(2 eta) ; (dz - k) w(0) = p(0)/(2 eta)                              (eq 24)
      gH = (part ? pH_im : pH_re) / (2.0 * eta);
      g0 = (part ? p0_im : p0_re) / (2.0 * eta);
    }
    const double beta_bc = par ? 0.5 * (gH + g0) : 0.5 * (gH - g0);
    const double Sc = chain_solve<NZ>(col, nullptr, VEC(10) + m, VEC(11) + m, VEC(12) + m, par, k, k2, inv_s, beta_bc, s_Bg[par * TM + m]);
    s_sum[(((1 + comp) * 2 + part) * 2 + par) * TM + m] = Sc;
  }
  __syncthreads();

  // ---------------- phase 6a: E_l = exp(-k z_l), z_l E_l at the nodes (C3); warp 0: correction coefficients
  for (int l = wid; l < NZ; l += NWARPS) {
    const double zl = s * (1.0 + T[Tab<NZ>::XI + l]);
    const double E = exp(-k * zl);
    VEC(6)[l * TM + m] = E;
    VEC(7)[l * TM + m] = zl * E;
  }
  if (wid == 0) {
    // wall data (eq 27 / (A3) with no slip, u_wall = 0): u_0 = -u_DP(z=0) = -(S_even - S_odd), u_H = -u_DP(z=H) = -(S_even + S_odd)
    double u0r[3], u0i[3], uHr[3], uHi[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double er = s_sum[(((1 + c) * 2 + 0) * 2 + 0) * TM + m], orr = s_sum[(((1 + c) * 2 + 0) * 2 + 1) * TM + m];
      const double ei = s_sum[(((1 + c) * 2 + 1) * 2 + 0) * TM + m], oi = s_sum[(((1 + c) * 2 + 1) * 2 + 1) * TM + m];
      u0r[c] = -(er - orr); u0i[c] = -(ei - oi); uHr[c] = -(er + orr); uHi[c] = -(ei + oi);
    }
    // coefficient layout: s_corr[((c*4 + basis)*2 + part)*TM + m], basis: 0 = z e^{-kz}, 1 = e^{-kz}, 2 = z e^{-k(H-z)}, 3 = e^{-k(H-z)}
    double cf[3][4][2];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int b = 0; b < 4; ++b) { cf[c][b][0] = 0.0; cf[c][b][1] = 0.0; }
    if (A.wall_mode == DP_BOTTOM_WALL) {
      // eqs 42-44: Q = i k w0 + kx u0 + ky v0 ; Wc = k w0 - i kx u0 - i ky v0
      const double Qr = -k * u0i[2] + kxt * u0r[0] + kyt * u0r[1], Qi = k * u0r[2] + kxt * u0i[0] + kyt * u0i[1];
      const double Wr = k * u0r[2] + kxt * u0i[0] + kyt * u0i[1], Wi = k * u0i[2] - kxt * u0r[0] - kyt * u0r[1];
      cf[0][0][0] = -(kxt / k) * Qr; cf[0][0][1] = -(kxt / k) * Qi;
      cf[1][0][0] = -(kyt / k) * Qr; cf[1][0][1] = -(kyt / k) * Qi;
      cf[2][0][0] = Wr; cf[2][0][1] = Wi;
#pragma unroll
      for (int c = 0; c < 3; ++c) { cf[c][1][0] = u0r[c]; cf[c][1][1] = u0i[c]; }
    } else {
      // App. A, no slip.  Unknowns [C0', D0', Cz, Dz] with C0' = C0/(2 eta), D0' = D0 e^{kH}/(2 eta) (basis e^{-k(H-z)}):
      // (A8b), (A8d), (A10a), (A10b) after eliminating Cx+e Dx, e Cx+Dx (and y) with (A8a), (A8c); e = e^{-kH}.
      const double e = exp(-k * A.H), H = A.H;
      const double g = (kxt * kxt + kyt * kyt) * H / k;
      double M[4][4] = {{0.0, 0.0, 1.0, e}, {H * e, H, e, 1.0}, {1.0, e, -k, k * e}, {e * (1.0 - g), 1.0 + g, -k * e, k}};
      double br[4] = {u0r[2], uHr[2], kxt * u0i[0] + kyt * u0i[1], kxt * uHi[0] + kyt * uHi[1]};
      double bi[4] = {u0i[2], uHi[2], -(kxt * u0r[0] + kyt * u0r[1]), -(kxt * uHr[0] + kyt * uHr[1])};
      solve4(M, br, bi);
      const double C0r = br[0], C0i = bi[0], D0r = br[1], D0i = bi[1];
      const double om = -expm1(-k * H) * (1.0 + e);       // 1 - e^2
#pragma unroll
      for (int c = 0; c < 2; ++c) {
        const double kc = c == 0 ? kxt : kyt, q = kc * H / k;
        // C_c + e D_c = u0 ; e C_c + D_c = uH + i q (e C0' - D0')
        const double r2r = uHr[c] - q * (e * C0i - D0i), r2i = uHi[c] + q * (e * C0r - D0r);
        cf[c][1][0] = (u0r[c] - e * r2r) / om; cf[c][1][1] = (u0i[c] - e * r2i) / om;
        cf[c][3][0] = (r2r - e * u0r[c]) / om; cf[c][3][1] = (r2i - e * u0i[c]) / om;
        // (A5): -i (k_c/k) C0' z e^{-kz} + i (k_c/k) D0' z e^{-k(H-z)}
        cf[c][0][0] = (kc / k) * C0i; cf[c][0][1] = -(kc / k) * C0r;
        cf[c][2][0] = -(kc / k) * D0i; cf[c][2][1] = (kc / k) * D0r;
      }
      // (A6): C0' z e^{-kz} + D0' z e^{-k(H-z)} + Cz e^{-kz} + Dz e^{-k(H-z)}
      cf[2][0][0] = C0r; cf[2][0][1] = C0i; cf[2][2][0] = D0r; cf[2][2][1] = D0i;
      cf[2][1][0] = br[2]; cf[2][1][1] = bi[2]; cf[2][3][0] = br[3]; cf[2][3][1] = bi[3];
    }
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int b = 0; b < 4; ++b) { s_corr[((c * 4 + b) * 2 + 0) * TM + m] = cf[c][b][0]; s_corr[((c * 4 + b) * 2 + 1) * TM + m] = cf[c][b][1]; }
  }
  __syncthreads();

  // ---------------- phase 6b: Chebyshev coefficients of E and zE (step 6)
  {
    double e[LH];
    const bool act = wid < 4;
    double* v = VEC(6 + (act ? wid >> 1 : 0)) + m;
    if (act) analysis_load<NZ>(v, wid & 1, e);
    __syncthreads();
    if (act) { if (wid & 1) analysis_compute<NZ, 1>(v, e); else analysis_compute<NZ, 0>(v, e); }
  }
  __syncthreads();

  // ---------------- phase 7: total coefficients = DP + correction;  T[z e^{-k(H-z)}]_n = (-1)^n (H e_n - ze_n), T[e^{-k(H-z)}]_n = (-1)^n e_n
  for (int n = wid; n < NZ; n += NWARPS) {
    const double en = VEC(6)[n * TM + m], zen = VEC(7)[n * TM + m];
    const double sgn = (n & 1) ? -1.0 : 1.0;
    const double b2 = sgn * (A.H * en - zen), b3 = sgn * en;
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int part = 0; part < 2; ++part) {
        double add = s_corr[((c * 4 + 0) * 2 + part) * TM + m] * zen + s_corr[((c * 4 + 1) * 2 + part) * TM + m] * en;
        if (A.wall_mode == DP_SLIT) add += s_corr[((c * 4 + 2) * 2 + part) * TM + m] * b2 + s_corr[((c * 4 + 3) * 2 + part) * TM + m] * b3;
        VEC(2 * c + part)[n * TM + m] += add;
      }
  }
  __syncthreads();

  // ---------------- phase 8: dz u, dz v of the TOTAL in coefficient space (reading G12) -> C3, C4
  if (A.omega) {
    const int comp = wid >> 2, part = (wid >> 1) & 1, par = wid & 1;     // 8 items = 8 warps
    deriv_sweep<NZ, false>(VEC(2 * comp + part) + m, VEC(6 + 2 * comp + part) + m, par, inv_s, 1.0);
  }
  __syncthreads();

  // ---------------- phase 9: synthesis back to the nodes
  {
    const int items = A.omega ? 10 : 6;
    for (int item = wid; item < items; item += NWARPS) synthesis_inplace<NZ>(VEC(item) + m);
  }
  __syncthreads();

  // ---------------- phase 10: (1/2) curl u (eq 11), scale by 1/(nx ny) for the unnormalised inverse FFT, store
  const double scl = 1.0 / ((double)A.nx * (double)A.ny);
  if (valid && !zero_mode) {
    for (int l = wid; l < NZ; l += NWARPS) {
      const int o = l * TM + m;
      const size_t off = ((size_t)l * A.ny + iy) * A.nkxp + ix;
      const double ur = VEC(0)[o], ui = VEC(1)[o], vr = VEC(2)[o], vi = VEC(3)[o], wr = VEC(4)[o], wi = VEC(5)[o];
      A.cplx[0 * A.cplx_field + off] = make_double2(ur * scl, ui * scl);
      A.cplx[1 * A.cplx_field + off] = make_double2(vr * scl, vi * scl);
      A.cplx[2 * A.cplx_field + off] = make_double2(wr * scl, wi * scl);
      if (A.omega) {
        const double dur = VEC(6)[o], dui = VEC(7)[o], dvr = VEC(8)[o], dvi = VEC(9)[o];
        A.cplx[3 * A.cplx_field + off] = make_double2(0.5 * (-kyt * wi - dvr) * scl, 0.5 * (kyt * wr - dvi) * scl);
        A.cplx[4 * A.cplx_field + off] = make_double2(0.5 * (dur + kxt * wi) * scl, 0.5 * (dui - kxt * wr) * scl);
        A.cplx[5 * A.cplx_field + off] = make_double2(-0.5 * (kxt * vi - kyt * ui) * scl, 0.5 * (kxt * vr - kyt * ur) * scl);
      }
    }
  }
#undef VEC
}

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
      for (int l = 0; l < nz; ++l) {
        double2 v = A.cplx[field * A.cplx_field + (size_t)l * A.ny * A.nkxp];
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
    const size_t off = (size_t)l * A.ny * A.nkxp;
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

template <int NZ> size_t solve_smem_bytes() { return sizeof(double) * ((size_t)NVEC * NZ * TM + 2 * TM + 16 * TM); }

template <int NZ> void host_tables(std::vector<double>& out) {
  typedef long double ld;
  const ld PI = 3.141592653589793238462643383279502884L;
  constexpr int N = NZ - 1, LH = NZ / 2;
  out.assign(Tab<NZ>::SIZE, 0.0);
  for (int n = 0; n <= N; ++n)
    for (int l = 0; l < LH; ++l) out[Tab<NZ>::CT + n * LH + l] = (double)cosl(PI * n * l / N);
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

template <int NZ> cudaError_t launch_nz(const SolveArgs& A, cudaStream_t st) {
  static bool attr = false;
  const size_t smem = solve_smem_bytes<NZ>();
  if (!attr) {
    cudaError_t e = cudaFuncSetAttribute(k_solve<NZ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr = true;
  }
  dim3 grid((A.nkx + TM - 1) / TM, A.ny);
  k_solve<NZ><<<grid, SOLVE_THREADS, smem, st>>>(A);
  return cudaGetLastError();
}

double* g_ct_full[3] = {nullptr, nullptr, nullptr};   // device cos tables for the k = 0 kernel (per compiled nz)
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
  const int slot = nz_slot(nz);
  if (!g_ct_full[slot]) {
    typedef long double ld;
    const ld PI = 3.141592653589793238462643383279502884L;
    std::vector<double> ct((size_t)nz * nz);
    for (int n = 0; n < nz; ++n) for (int l = 0; l < nz; ++l) ct[(size_t)n * nz + l] = (double)cosl(PI * n * l / (nz - 1));
    e = cudaMalloc(&g_ct_full[slot], sizeof(double) * ct.size());
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(g_ct_full[slot], ct.data(), sizeof(double) * ct.size(), cudaMemcpyHostToDevice);
  }
  return e;
}

cudaError_t dp_launch_solve(dp_plan* P, bool with_torque_field, bool want_omega, cudaStream_t st) {
  SolveArgs A;
  A.cplx = P->d_cplx; A.cplx_field = P->cplx_field;
  A.nx = P->p.nx; A.ny = P->p.ny; A.nkx = P->nkx; A.nkxp = P->nkxp;
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
  k_zero_mode<<<1, 64, 0, st>>>(A, P->p.nz, g_ct_full[nz_slot(P->p.nz)]);
  return cudaGetLastError();
}
