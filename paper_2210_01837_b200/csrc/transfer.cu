// transfer.cu — particle <-> grid kernels: binning (a0), spreading (a1, a2; paper step 1), interpolation (a12; step 8).
//
// Step 1 (eqs 7, 9, 53, 54): f(x_g) = sum_j F_j Delta_M^W(x_g - r_j), t(x_g) = sum_j tau_j Delta_D^W(x_g - r_j)
//   Delta^W = phi(x)phi(y)[phi(z - z_j) - phi(z + z_j) - (slit) phi(z - (2H - z_j))]
// Step 8 (eqs 10, 11): U_j = sum_g u(x_g) Delta_M^W(x_g - r_j) h^2 (H/2) w_l, Omega_j likewise with Delta_D^W.
//
// Kernel-derivative torque mode (dp_params.torque_mode = 1; the paper's "second way", footnotes 47-48): the torques
// are spread into the SAME three fields as the forces, f += (1/2) G x tau with G = grad_x Delta_D^W =
// (phi'(x)phi(y)zeta(l), phi(x)phi'(y)zeta(l), phi(x)phi(y)zeta'(l)), and Omega_j = (1/2) sum_g (u(x_g) x G(x_g)) h^2 (H/2) w_l is
// gathered from the velocity field itself (eq 11 integrated by parts), so only three fields are transformed each way.
//
// B200 design: particles are counting-sorted by the xy tile (16 x 4 grid columns) that contains the origin of
// their w x w footprint.  One CTA owns one tile of one field triple and gathers every footprint that touches it into
// per-thread register accumulators (each thread owns one column and a fixed residue class of the plane index, so no
// atomics and no conflicts), then stores the tile to HBM once in 128-byte row segments — every grid value is written
// exactly once, zeros included, so there is no memset pass and no global atomic.
#include "common.cuh"

namespace {

constexpr int TX = DP_TILE_X, TY = DP_TILE_Y;
// z residue classes per grid column = threads per column of the spread kernels, by compiled nz: with the pipelined kernel hiding the global
// latency, ONE thread per column (all of its planes in registers: no per-column set-up repeated by several threads) is fastest up to nz = 32
// (measured at cfg 5: 4.7 ms against 5.0 with two and 6.0 with four); larger nz need two to keep the accumulators in registers.
// ZSPLIT / SPREAD_THREADS are usable wherever a template parameter (or macro argument) NZ is in scope.
#define DP_ZSPLIT_OF(NZ) ((NZ) <= 32 ? 1 : 2)
#define ZSPLIT (DP_ZSPLIT_OF(NZ))
#define SPREAD_THREADS (TX * TY * ZSPLIT)
#define DP_PCH 40
constexpr int PCH = DP_PCH;                     // candidate particles staged per chunk
constexpr int MAXB = 6;                         // origin bins per direction that can reach a tile (w <= 8, TY = 4)
constexpr int MAXR = 2 * MAXB;                  // candidate ranges per tile: one per bin row, two when the x range wraps
#define MAXKEEP SPREAD_THREADS                  // survivors of one block of candidates

struct GridGeom {
  int nx, ny, nz, w, wall_mode, nbx, nby;
  double Lx, Ly, H, h, alpha;
};

__device__ __forceinline__ int origin_cell(double xw, double alpha, double h, int n) {
  // first node of the footprint: i0 = ceil((x - alpha)/h), nodes i0 .. i0+w-1 (reading G6)
  int i0 = (int)ceil((xw - alpha) / h);
  i0 %= n;
  return i0 < 0 ? i0 + n : i0;
}

// Bins (of width T, the last one possibly narrower) that hold the origin columns o with o..o+w-1 (cyclic, period n)
// reaching the tile [X0, X0+Teff): the cyclic range [X0-w+1, X0+Teff-1], of length Teff+w-1 <= n (checked at create).
__device__ __forceinline__ int origin_bins(int X0, int Teff, int T, int w, int n, int* out) {
  int o = X0 - (w - 1); o %= n; if (o < 0) o += n;
  int left = Teff + w - 1, cnt = 0;
  while (left > 0 && cnt < MAXB) {
    int b = o / T, bend = min((b + 1) * T, n);
    out[cnt++] = b;
    left -= bend - o;
    o = bend == n ? 0 : bend;
  }
  return cnt;
}

// ---------------------------------------------------------------------------------------------- z weights
// zeta(l; z_p) = phi(z_l - z_p) - phi(z_l + z_p) - [slit] phi(z_l - (2H - z_p))   (eq 9)
// phi(s) of eq 54 with 1/alpha and 1/Z precomputed (support test |s| <= alpha inclusive, reading G6)
__device__ __forceinline__ double es_phi(double s, double inv_alpha, double beta, double inv_Z) {
  const double q = s * inv_alpha;
  if (!(fabs(q) <= 1.0)) return 0.0;
  double r = 1.0 - q * q; r = r < 0.0 ? 0.0 : r;
  return exp(beta * (sqrt(r) - 1.0)) * inv_Z;
}
__device__ __forceinline__ double zeta_weight(double zl, double zp, double H, int wall_mode, double inv_alpha, double beta, double inv_Z) {
  double v = es_phi(zl - zp, inv_alpha, beta, inv_Z) - es_phi(zl + zp, inv_alpha, beta, inv_Z);
  if (wall_mode == DP_SLIT) v -= es_phi(zl - (2.0 * H - zp), inv_alpha, beta, inv_Z);
  return v;
}
// truncated derivative of eq 54's kernel (footnote 47): phi'(s) = -(beta s/alpha^2) phi(s)/sqrt(1-(s/alpha)^2) for
// |s| <= ucut alpha, 0 beyond (ucut: where |phi'| is smallest before it blows up at the edge of the support, see plan.cu)
__device__ __forceinline__ double es_dphi(double s, double inv_alpha, double beta, double inv_Z, double ucut) {
  const double q = s * inv_alpha;
  if (!(fabs(q) <= ucut)) return 0.0;
  const double sr = sqrt(1.0 - q * q);
  return -(beta * q * inv_alpha) * exp(beta * (sr - 1.0)) * inv_Z / sr;
}
// zeta'(l; z_p) = d/dz [phi(z - z_p) - phi(z + z_p) - [slit] phi(z - (2H - z_p))] at z = z_l: the exact z-derivative of eq 9,
// which vanishes with the particle's height (footnote 48; reading G19)
__device__ __forceinline__ double dzeta_weight(double zl, double zp, double H, int wall_mode, double inv_alpha, double beta, double inv_Z, double ucut) {
  double v = es_dphi(zl - zp, inv_alpha, beta, inv_Z, ucut) - es_dphi(zl + zp, inv_alpha, beta, inv_Z, ucut);
  if (wall_mode == DP_SLIT) v -= es_dphi(zl - (2.0 * H - zp), inv_alpha, beta, inv_Z, ucut);
  return v;
}
// node range with z_l in [max(0, zp - alpha), min(H, zp + alpha)] (nodes decrease with l); covers every image term
__device__ __forceinline__ void z_range(const double* zn, int nz, double zp, double alpha, double H, int& lmin, int& lmax) {
  double hi = zp + alpha, lo = zp - alpha;
  int a = 0, b = nz - 1;
  while (a < nz && zn[a] > hi) ++a;
  while (b >= 0 && zn[b] < lo) --b;
  lmin = a; lmax = b;
}

// ---------------------------------------------------------------------------------------------- binning
__global__ void k_bin_count(int n, const double* __restrict__ pos, GridGeom g, int* __restrict__ bin_of,
                            int* __restrict__ slot_of, int* __restrict__ bin_count, int* __restrict__ flag) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  double x = pos[3 * (size_t)p], y = pos[3 * (size_t)p + 1], z = pos[3 * (size_t)p + 2];
  bool ok = (z >= 0.0) && (z <= g.H) && (g.wall_mode == DP_SLIT || z + g.alpha <= g.H) && isfinite(x) && isfinite(y);
  int b = 0;
  if (ok) {
    double xw = x - floor(x / g.Lx) * g.Lx, yw = y - floor(y / g.Ly) * g.Ly;
    int i0 = origin_cell(xw, g.alpha, g.h, g.nx), j0 = origin_cell(yw, g.alpha, g.h, g.ny);
    b = (j0 / TY) * g.nbx + (i0 / TX);
  } else {
    atomicOr(flag, 1);
  }
  bin_of[p] = b;
  slot_of[p] = atomicAdd(&bin_count[b], 1);
}

// exclusive scan of bin_count -> bin_start[0..nbins] in two launches: k_scan_local scans chunks of SCAN_CHUNK bins (one CTA each, eight
// consecutive bins per thread) and leaves each chunk's total in block_sum; k_scan_add adds the totals of the preceding chunks
constexpr int SCAN_THREADS = 1024, SCAN_E = 8, SCAN_CHUNK = SCAN_THREADS * SCAN_E;
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_local(int nbins, const int* __restrict__ cnt, int* __restrict__ start, int* __restrict__ block_sum) {
  __shared__ int warp_sums[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int i0 = blockIdx.x * SCAN_CHUNK + threadIdx.x * SCAN_E;
  int v[SCAN_E], tot = 0;
#pragma unroll
  for (int e = 0; e < SCAN_E; ++e) { v[e] = (i0 + e < nbins) ? cnt[i0 + e] : 0; tot += v[e]; }
  int s = tot;
  for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += t; }
  if (lane == 31) warp_sums[wid] = s;
  __syncthreads();
  if (wid == 0) {
    int ws = warp_sums[lane];
    for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, ws, o); if (lane >= o) ws += t; }
    warp_sums[lane] = ws;
  }
  __syncthreads();
  int run = (wid > 0 ? warp_sums[wid - 1] : 0) + s - tot;                 // exclusive prefix of this thread's first bin within the chunk
#pragma unroll
  for (int e = 0; e < SCAN_E; ++e) { if (i0 + e < nbins) start[i0 + e] = run; run += v[e]; }
  if (threadIdx.x == SCAN_THREADS - 1) block_sum[blockIdx.x] = run;
}
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_add(int nbins, int nblocks, int* __restrict__ start, const int* __restrict__ block_sum) {
  __shared__ int s_off, s_part[32];
  // offset of this chunk = sum of the totals of the chunks before it (a few dozen values: one warp-shuffle reduction per 1024)
  int acc = 0;
  for (int b = threadIdx.x; b < (int)blockIdx.x; b += SCAN_THREADS) acc += block_sum[b];
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) { int t = 0; for (int w = 0; w < SCAN_THREADS / 32; ++w) t += s_part[w]; s_off = t; }
  __syncthreads();
  const int off = s_off;
  const int i0 = blockIdx.x * SCAN_CHUNK + threadIdx.x * SCAN_E;
#pragma unroll
  for (int e = 0; e < SCAN_E; ++e) if (i0 + e < nbins) start[i0 + e] += off;
  if ((int)blockIdx.x == nblocks - 1 && threadIdx.x == 0) start[nbins] = off + block_sum[blockIdx.x];
}

__global__ void k_bin_scatter(int n, const double* __restrict__ pos, const double* __restrict__ force,
                              const double* __restrict__ torque, GridGeom g, const int* __restrict__ bin_of,
                              const int* __restrict__ slot_of, const int* __restrict__ bin_start, const double* __restrict__ znodes,
                              int* __restrict__ perm, int4* __restrict__ meta, double* __restrict__ pos_s, double* __restrict__ frc_s,
                              double* __restrict__ trq_s, int* __restrict__ lmin_all) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  int my_lmin = 0x7fffffff;
  if (p < n) {
  int d = bin_start[bin_of[p]] + slot_of[p];
  perm[d] = p;
  double x = pos[3 * (size_t)p], y = pos[3 * (size_t)p + 1], z = pos[3 * (size_t)p + 2];
  bool ok = (z >= 0.0) && (z <= g.H) && (g.wall_mode == DP_SLIT || z + g.alpha <= g.H) && isfinite(x) && isfinite(y);
  double xw = 0.0, yw = 0.0;
  if (ok) { xw = x - floor(x / g.Lx) * g.Lx; yw = y - floor(y / g.Ly) * g.Ly; }
  pos_s[3 * (size_t)d] = xw; pos_s[3 * (size_t)d + 1] = yw; pos_s[3 * (size_t)d + 2] = ok ? z : -1.0;   // z < 0: skipped
  // footprint record: wrapped origin node (i0, j0) and plane range [lmin, lmax]; lmin > lmax marks a skipped particle
  int4 m = make_int4(0, 0, 1, 0);
  if (ok) {
    m.x = origin_cell(xw, g.alpha, g.h, g.nx); m.y = origin_cell(yw, g.alpha, g.h, g.ny);
    z_range(znodes, g.nz, z, g.alpha, g.H, m.z, m.w);
  }
  meta[d] = m;
  for (int c = 0; c < 3; ++c) {
    if (frc_s) frc_s[3 * (size_t)d + c] = force ? force[3 * (size_t)p + c] : 0.0;
    if (trq_s) trq_s[3 * (size_t)d + c] = torque ? torque[3 * (size_t)p + c] : 0.0;
  }
  if (ok && m.z <= m.w) my_lmin = m.z;
  }
  // highest plane (lowest index) any footprint touches: one atomic per warp
  my_lmin = __reduce_min_sync(0xffffffffu, my_lmin);
  if ((threadIdx.x & 31) == 0 && my_lmin != 0x7fffffff) atomicMin(lmin_all, my_lmin);
}

// ---------------------------------------------------------------------------------------------- 1-D ES weights
// One record per particle and envelope (0: Delta_M, 1: Delta_D, 2 (kernel-derivative torque mode): the derivatives of record 1,
// phi'(x), phi'(y), zeta'(l)), in sorted order, evaluated once per product and used by
// both spreading and interpolation:  rec[0..7] = phi(x_{i0+a} - x), rec[8..15] = phi(y_{j0+b} - y), rec[16+l] = zeta(l; z)
// (eqs 9, 54).  One thread per record entry.
struct WeightArgs {
  GridGeom g;
  const double* pos_s;
  const int4* meta;
  const double* znodes;
  double beta[3], inv_Z[3];  // record 2 uses the dipole envelope's beta and Z
  double inv_alpha;
  double ucut;               // truncation point of phi' (record 2)
  double* wrec;              // [nrec][cap][16 + nz]
  size_t cap;
};

// One warp per particle, all of its records.  Only about 22 of the 16 + nz entries of a record are not zero (w + w in x, y and the planes
// lmin..lmax in z), and every evaluation of the kernel costs an exp and a square root: the warp first stores zeros over the whole
// record, then lanes 0-7 take the x entries, 8-15 the y entries and lanes 16-31 the planes lmin, lmin + 1, ... sixteen at a time, so a
// warp evaluates the kernel once (plus once per image term of eq 9 that reaches some plane) instead of once per 32 record entries.
#define DP_WEIGHT_WARPS 8
constexpr int WEIGHT_WARPS = DP_WEIGHT_WARPS;
__global__ void __launch_bounds__(WEIGHT_WARPS * 32) k_weights(int n, WeightArgs A, int nrec) {
  const GridGeom& g = A.g;
  const int wrec = 2 * DP_MAX_W + g.nz;
  const int lane = threadIdx.x & 31, p = blockIdx.x * WEIGHT_WARPS + (threadIdx.x >> 5);
  if (p >= n) return;
  const int4 m = A.meta[p];
  const double inv_alpha = A.inv_alpha;
  // the particle's coordinate this lane works with: x for lanes 0-7, y for 8-15, z for the rest (one load for all of its records)
  const double c = A.pos_s[3 * (size_t)p + (lane < DP_MAX_W ? 0 : (lane < 2 * DP_MAX_W ? 1 : 2))];
  for (int k = 0; k < nrec; ++k) {
    double* rec = A.wrec + ((size_t)k * A.cap + p) * wrec;
    for (int e = lane; e < wrec; e += 32) rec[e] = 0.0;
  }
  if (m.z > m.w) return;                                         // skipped particle: all-zero records
  __syncwarp();
  const int a = lane & (DP_MAX_W - 1);
  const double i0 = ceil((c - g.alpha) / g.h);                   // unwrapped origin: distances use the unwrapped node (same expression as origin_cell)
  const bool is_xy = lane < 2 * DP_MAX_W;
  const double far = 4.0 * g.alpha;                              // a distance outside every support
  for (int k = 0; k < nrec; ++k) {
    const double beta = A.beta[k], inv_Z = A.inv_Z[k];
    double* rec = A.wrec + ((size_t)k * A.cap + p) * wrec;
    // every lane evaluates the kernel ONCE per round at its own distance (x, y entries: node minus particle; z entries: z_l - z_p, sixteen
    // planes per round); the image terms of eq 9 follow for the z lanes only where some lane of the warp is inside their support
    for (int l0 = m.z; l0 <= m.w || l0 == m.z; l0 += 32 - 2 * DP_MAX_W) {
      const int l = l0 + (lane - 2 * DP_MAX_W);
      const bool zon = !is_xy && l <= m.w, xyon = is_xy && a < g.w && l0 == m.z;
      const double zl = zon ? A.znodes[l] : 0.0;
      const double s1 = xyon ? (i0 + a) * g.h - c : (zon ? zl - c : far);
      const double s2 = zon ? zl + c : far, s3 = (zon && g.wall_mode == DP_SLIT) ? zl - (2.0 * g.H - c) : far;
      double v;
      if (k < 2) {
        v = es_phi(s1, inv_alpha, beta, inv_Z);
        if (__any_sync(0xffffffffu, fabs(s2) <= g.alpha)) v -= es_phi(s2, inv_alpha, beta, inv_Z);
        if (__any_sync(0xffffffffu, fabs(s3) <= g.alpha)) v -= es_phi(s3, inv_alpha, beta, inv_Z);
      } else {
        v = es_dphi(s1, inv_alpha, beta, inv_Z, A.ucut);
        if (__any_sync(0xffffffffu, fabs(s2) <= g.alpha)) v -= es_dphi(s2, inv_alpha, beta, inv_Z, A.ucut);
        if (__any_sync(0xffffffffu, fabs(s3) <= g.alpha)) v -= es_dphi(s3, inv_alpha, beta, inv_Z, A.ucut);
      }
      if (xyon) rec[lane] = v;
      else if (zon) rec[2 * DP_MAX_W + l] = v;
    }
  }
}

// ---------------------------------------------------------------------------------------------- spread
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async16(double* smem_dst, const double* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_commit_only() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_only() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all_groups() { asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory"); }

struct SpreadArgs {
  GridGeom g;
  const double* val_s[2];    // forces, torques (sorted)
  int field0[2];             // first output field of each group
  const int* bin_start;
  const int4* meta;          // sorted footprint records (i0, j0, lmin, lmax)
  const double* wrec;        // sorted weight records
  size_t cap;
  double* grid;
  size_t real_field;
  const int* lmin;           // planes l < *lmin hold no force: not stored (the forward FFT passes skip them)
};

// One CTA = one tile of TX x TY grid columns of one field triple.  Thread (ti, tj, tz) owns column (ti, tj) and the
// planes l = ZSPLIT*li + tz; its 3*NZ/ZSPLIT partial sums live in registers for the whole kernel, so there is no
// shared-memory tile, no atomic and no memset.  The candidates (the bins whose footprints can reach the tile, merged
// into contiguous ranges of the sorted arrays) are culled by their footprint records; the survivors are staged in shared
// memory with their weight records; every thread adds the particles covering its column; each grid value is stored to HBM
// exactly once (128-byte row segments per warp).  Dependent global round trips per CTA: bin_start -> footprint records ->
// weight records -> stores.
// GT = double, or float for the optional fp32 variant (accumulators and grid in fp32; the weight records stay fp64 and are
// rounded when they are used).
// MODE 0: field triple blockIdx.z (0: forces with Delta_M, 1: torques with Delta_D) gets sum_j val_j S(j; g)   (eq 7 without the curl,
//         which the solve kernel takes in Fourier-Chebyshev space);
// MODE 1 (kernel-derivative torques): ONE triple f = sum_j [F_j S_M(j; g) + (1/2) G_j(g) x tau_j], three records per candidate.
#define DP_SPREAD_MINB (NZ <= 32 ? 4 : 2)
// staged candidates of one chunk: weight records (zero padded to whole z residue classes), values, footprint records
template <int NZ, int MODE> struct SpreadBuf {
  static constexpr int NL = (NZ + ZSPLIT - 1) / ZSPLIT;
  static constexpr int WREC = 2 * DP_MAX_W + NZ;                 // record length in global memory
  static constexpr int WS = 2 * DP_MAX_W + NL * ZSPLIT;          // staged record length
  static constexpr int NREC = MODE ? 3 : 1;
  static constexpr int PC = MODE ? PCH / 2 : PCH;                // candidates per chunk
  static constexpr int NV = MODE ? 6 : 3;
  double w[PC][NREC][WS];
  double val[PC][NV];
  int4 meta[PC];                                                 // i0, j0 (wrapped origin node), lmin, lmax
};

// every thread adds the nl staged particles that cover its column (gi, gj) to its own planes l = ZSPLIT li + tz
template <int NZ, class GT, int MODE>
__device__ __forceinline__ void accumulate_chunk(GT (&acc)[(NZ + ZSPLIT - 1) / ZSPLIT][3], const SpreadBuf<NZ, MODE>& B, int nl, const GridGeom& g, int gi, int gj, int tz,
                                                 bool in_grid) {
  constexpr int NL = SpreadBuf<NZ, MODE>::NL, NV = SpreadBuf<NZ, MODE>::NV;
  const int w = g.w;
  if (in_grid) {
    for (int q = 0; q < nl; ++q) {
      const int4 m = B.meta[q];
      int a = gi - m.x; if (a < 0) a += g.nx;
      int bb = gj - m.y; if (bb < 0) bb += g.ny;
      if (a < w && bb < w) {
        if (MODE == 0) {
          const GT wxy = (GT)B.w[q][0][a] * (GT)B.w[q][0][DP_MAX_W + bb];
          const GT v0 = (GT)B.val[q][0] * wxy, v1 = (GT)B.val[q][1] * wxy, v2 = (GT)B.val[q][2] * wxy;
          const double* zt = &B.w[q][0][2 * DP_MAX_W + tz];
          // zeta vanishes outside [lmin, lmax]: skipping a half of the planes that lies outside is exact
          if (m.z < ZSPLIT * (NL / 2)) {
#pragma unroll
            for (int li = 0; li < NL / 2; ++li) {
              const GT z = (GT)zt[ZSPLIT * li];
              acc[li][0] = fma(v0, z, acc[li][0]); acc[li][1] = fma(v1, z, acc[li][1]); acc[li][2] = fma(v2, z, acc[li][2]);
            }
          }
          if (m.w >= ZSPLIT * (NL / 2)) {
#pragma unroll
            for (int li = NL / 2; li < NL; ++li) {
              const GT z = (GT)zt[ZSPLIT * li];
              acc[li][0] = fma(v0, z, acc[li][0]); acc[li][1] = fma(v1, z, acc[li][1]); acc[li][2] = fma(v2, z, acc[li][2]);
            }
          }
        } else {
          const double* wM = B.w[q][0]; const double* wD = B.w[q][MODE ? 1 : 0]; const double* wG = B.w[q][MODE ? 2 : 0];
          const GT pM = (GT)wM[a] * (GT)wM[DP_MAX_W + bb];
          const GT c0f = (GT)B.val[q][0] * pM, c1f = (GT)B.val[q][1] * pM, c2f = (GT)B.val[q][2] * pM;     // x zeta_M(l)
          const GT tx = (GT)B.val[q][NV - 3], ty = (GT)B.val[q][NV - 2], tzq = (GT)B.val[q][NV - 1];
          const GT pxy = (GT)wD[a] * (GT)wD[DP_MAX_W + bb];                   // phi(x) phi(y)
          const GT dxy = (GT)wG[a] * (GT)wD[DP_MAX_W + bb];                   // phi'(x) phi(y)
          const GT xdy = (GT)wD[a] * (GT)wG[DP_MAX_W + bb];                   // phi(x) phi'(y)
          // (1/2) G x tau with G = (dxy zeta, xdy zeta, pxy zeta'):  coefficients of zeta_D(l) and of zeta_D'(l)
          const GT a0 = (GT)0.5 * tzq * xdy, a1 = -(GT)0.5 * tzq * dxy, a2 = (GT)0.5 * (ty * dxy - tx * xdy);
          const GT b0 = -(GT)0.5 * ty * pxy, b1 = (GT)0.5 * tx * pxy;
          const double* zm = &wM[2 * DP_MAX_W + tz]; const double* zd = &wD[2 * DP_MAX_W + tz]; const double* zg = &wG[2 * DP_MAX_W + tz];
          if (m.z < ZSPLIT * (NL / 2)) {
#pragma unroll
            for (int li = 0; li < NL / 2; ++li) {
              const GT zM = (GT)zm[ZSPLIT * li], zD = (GT)zd[ZSPLIT * li], zG = (GT)zg[ZSPLIT * li];
              acc[li][0] = fma(c0f, zM, fma(a0, zD, fma(b0, zG, acc[li][0])));
              acc[li][1] = fma(c1f, zM, fma(a1, zD, fma(b1, zG, acc[li][1])));
              acc[li][2] = fma(c2f, zM, fma(a2, zD, acc[li][2]));
            }
          }
          if (m.w >= ZSPLIT * (NL / 2)) {
#pragma unroll
            for (int li = NL / 2; li < NL; ++li) {
              const GT zM = (GT)zm[ZSPLIT * li], zD = (GT)zd[ZSPLIT * li], zG = (GT)zg[ZSPLIT * li];
              acc[li][0] = fma(c0f, zM, fma(a0, zD, fma(b0, zG, acc[li][0])));
              acc[li][1] = fma(c1f, zM, fma(a1, zD, fma(b1, zG, acc[li][1])));
              acc[li][2] = fma(c2f, zM, fma(a2, zD, acc[li][2]));
            }
          }
        }
      }
    }
  }
}

// every grid value of the tile's planes that can hold force is written exactly once
template <int NZ, class GT>
__device__ __forceinline__ void store_tile(const GT (&acc)[(NZ + ZSPLIT - 1) / ZSPLIT][3], const SpreadArgs& A, const GridGeom& g, int grp, int gi, int gj, int tz, bool in_grid) {
  constexpr int NL = (NZ + ZSPLIT - 1) / ZSPLIT;
  if (in_grid) {
    const int lm = __ldg(A.lmin);
    GT* dst = reinterpret_cast<GT*>(A.grid) + (size_t)A.field0[grp] * A.real_field + ((size_t)tz * g.ny + gj) * g.nx + gi;
    const size_t step = (size_t)ZSPLIT * g.ny * g.nx;             // from plane l to plane l + ZSPLIT
#pragma unroll
    for (int li = 0; li < NL; ++li) {
      const int l = ZSPLIT * li + tz;
      if (l >= lm && l < NZ) {
#pragma unroll
        for (int c = 0; c < 3; ++c) dst[c * A.real_field] = acc[li][c];
      }
      dst += step;
    }
  }

}

// With a tile list (ov_tiles, *ov_count) the CTAs walk that list instead of taking the tile from blockIdx: the tiles the pipelined
// kernel below leaves to this one (more survivors than a staged chunk holds).
template <int NZ, class GT, int MODE>
__global__ void __launch_bounds__(SPREAD_THREADS, DP_SPREAD_MINB) k_spread(SpreadArgs A, const int* __restrict__ ov_tiles, const int* __restrict__ ov_count) {
  typedef SpreadBuf<NZ, MODE> SB;
  constexpr int NL = SB::NL, WREC = SB::WREC, WS = SB::WS, NREC = SB::NREC, PC = SB::PC;
  __shared__ __align__(16) SB B;
  __shared__ int s_rbeg[MAXR], s_roff[MAXR + 1];   // candidate ranges in the sorted arrays; prefix sums of their lengths
  __shared__ int s_keep[MAXKEEP];             // candidates whose footprint really touches the tile
  __shared__ int s_nkeep;

  const GridGeom& g = A.g;
  const int w = g.w;
  const int grp = blockIdx.z;
  const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const int ti = t % TX, tj = (t / TX) % TY, tz = t / (TX * TY);
  const int nlist = ov_tiles ? __ldg(ov_count) : 1;
  for (int it = ov_tiles ? (int)blockIdx.x : 0; it < nlist; it += ov_tiles ? (int)gridDim.x : 1) {
  const int tile = ov_tiles ? __ldg(ov_tiles + it) : -1;
  const int X0 = (tile >= 0 ? tile % g.nbx : (int)blockIdx.x) * TX, Y0 = (tile >= 0 ? tile / g.nbx : (int)blockIdx.y) * TY;
  const int gi = X0 + ti, gj = Y0 + tj;
  const bool in_grid = gi < g.nx && gj < g.ny;

  GT acc[NL][3];
#pragma unroll
  for (int li = 0; li < NL; ++li) { acc[li][0] = 0; acc[li][1] = 0; acc[li][2] = 0; }

  // bins whose footprints can reach this tile: origin columns in the cyclic range [X0-w+1, X0+TXeff-1] (same in y);
  // the x-bins of one bin row are consecutive in memory, so each row gives one range (two when the range wraps in x)
  if (wid == 0) {
    int o = X0 - (w - 1); o %= g.nx; if (o < 0) o += g.nx;
    const int len = min(TX, g.nx - X0) + w - 1;                 // <= nx (checked at create)
    const int b0 = o / TX, b1 = (o + len - 1 < g.nx) ? (o + len - 1) / TX : g.nbx - 1;
    const int wrap_b1 = (o + len - 1 < g.nx) ? -1 : (o + len - 1 - g.nx) / TX;     // second piece: bins 0 .. wrap_b1
    int bys[MAXB];
    const int ncy = origin_bins(Y0, min(TY, g.ny - Y0), TY, w, g.ny, bys);
    const int per_row = wrap_b1 >= 0 ? 2 : 1;
    const int nr = ncy * per_row;
    int beg = 0, cnt = 0;
    if (lane < nr) {
      const int row = bys[lane / per_row], piece = lane % per_row;
      const int ba = piece == 0 ? b0 : 0, bb = piece == 0 ? b1 : min(wrap_b1, b0 - 1);
      beg = A.bin_start[row * g.nbx + ba];
      cnt = bb >= ba ? A.bin_start[row * g.nbx + bb + 1] - beg : 0;
    }
    int incl = cnt;                                           // inclusive scan over the (<= MAXR) ranges
#pragma unroll
    for (int o2 = 1; o2 < 16; o2 <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o2); if (lane >= o2) incl += v; }
    if (lane < MAXR) { s_rbeg[lane] = beg; s_roff[lane + 1] = incl; }
    if (lane == 0) s_roff[0] = 0;
  }
  if (t == 0) s_nkeep = 0;
  __syncthreads();
  const int total = s_roff[MAXR];

  // Cull: the ranges hold every particle whose footprint ORIGIN lies in a bin that can reach the tile (2-3 times as many as
  // really touch it).  Blocks of 256 candidates: one pass over their footprint records keeps the ones whose w x w footprint
  // intersects the tile's columns (warp ballot + one shared-memory counter update per warp; the order of the survivors, hence
  // the summation order, is not fixed), then the survivors are staged with their weight records in chunks of PC and every
  // thread adds the ones covering its column to its own planes.
  const int TXe = min(TX, g.nx - X0), TYe = min(TY, g.ny - Y0);
  for (int blk = 0; blk < total; blk += SPREAD_THREADS) {
    {
      const int c = blk + t;
      bool keep = false;
      int src = 0;
      if (c < total) {
        int r = 0;
#pragma unroll
        for (int q = 1; q < MAXR; ++q) r += (c >= s_roff[q]) ? 1 : 0;
        src = s_rbeg[r] + (c - s_roff[r]);
        const int4 m = A.meta[src];
        int dx = X0 - m.x; if (dx < 0) dx += g.nx;          // tile start seen from the footprint origin
        int ex = m.x - X0; if (ex < 0) ex += g.nx;          // footprint origin seen from the tile start
        int dy = Y0 - m.y; if (dy < 0) dy += g.ny;
        int ey = m.y - Y0; if (ey < 0) ey += g.ny;
        keep = (m.z <= m.w) && (dx < w || ex < TXe) && (dy < w || ey < TYe);
      }
      const unsigned bal = __ballot_sync(0xffffffffu, keep);
      int base = 0;
      if (lane == 0 && bal) base = atomicAdd(&s_nkeep, __popc(bal));
      base = __shfl_sync(0xffffffffu, base, 0);
      if (keep) s_keep[base + __popc(bal & ((1u << lane) - 1))] = src;
    }
    __syncthreads();
    const int nkeep = s_nkeep;
    for (int c0 = 0; c0 < nkeep; c0 += PC) {
      const int nl = min(PC, nkeep - c0);
      if (t < nl) {
        const int p = s_keep[c0 + t];
        B.meta[t] = A.meta[p];
        if (MODE) {
#pragma unroll
          for (int c = 0; c < 3; ++c) { B.val[t][c] = A.val_s[0][3 * (size_t)p + c]; B.val[t][3 + c] = A.val_s[1][3 * (size_t)p + c]; }
        } else {
          const double* __restrict__ val = A.val_s[grp];
          B.val[t][0] = val[3 * (size_t)p]; B.val[t][1] = val[3 * (size_t)p + 1]; B.val[t][2] = val[3 * (size_t)p + 2];
        }
      }
      // the weight records travel as asynchronous 8-byte copies: all of a thread's entries are in flight at once (one round of
      // global latency per chunk instead of one per two entries)
      // (16 bytes per copy where the record length is even, i.e. every record starts on a 16-byte boundary)
      if constexpr (WREC % 2 == 0) {
        constexpr int WH = WS / 2;
        for (int i = t; i < nl * NREC * WH; i += SPREAD_THREADS) {
          const int q = i / (NREC * WH), rem = i - q * (NREC * WH), k = rem / WH, e = 2 * (rem - k * WH);
          const int kk = MODE ? k : grp;
          if (e < WREC) cp_async16(&B.w[q][k][e], A.wrec + ((size_t)kk * A.cap + s_keep[c0 + q]) * WREC + e);
          else { B.w[q][k][e] = 0.0; B.w[q][k][e + 1] = 0.0; }
        }
      } else {
        for (int i = t; i < nl * NREC * WS; i += SPREAD_THREADS) {
          const int q = i / (NREC * WS), rem = i - q * (NREC * WS), k = rem / WS, e = rem - k * WS;
          const int kk = MODE ? k : grp;
          if (e < WREC) cp_async8(&B.w[q][k][e], A.wrec + ((size_t)kk * A.cap + s_keep[c0 + q]) * WREC + e);
          else B.w[q][k][e] = 0.0;
        }
      }
      cp_async_wait_all_groups();
      __syncthreads();
      accumulate_chunk<NZ, GT, MODE>(acc, B, nl, g, gi, gj, tz, in_grid);
      __syncthreads();
    }
    if (t == 0) s_nkeep = 0;
    __syncthreads();
  }
  store_tile<NZ, GT>(acc, A, g, grp, gi, gj, tz, in_grid);
  __syncthreads();                             // the shared state is reused by the next tile of the list
  }
}

// ---------------------------------------------------------------------------------------------- spread, pipelined
// Per-tile survivor lists, built once per product by one warp per tile (k_tile_lists): the particles whose w x w footprint touches
// the tile's columns, at most LMAX stored, the true count beside them; tiles with more survivors than a staged chunk holds go to an
// overflow list that k_spread (above) works through.
constexpr int LMAX = PCH;
constexpr int LIST_WARPS = 8;
__global__ void __launch_bounds__(LIST_WARPS * 32) k_tile_lists(GridGeom g, const int* __restrict__ bin_start, const int4* __restrict__ meta, int pc_limit,
                                                                  int* __restrict__ tile_cnt, int* __restrict__ tile_list, int* __restrict__ ov_tiles, int* __restrict__ ov_count) {
  const int lane = threadIdx.x & 31, tile = blockIdx.x * LIST_WARPS + (threadIdx.x >> 5);
  if (tile >= g.nbx * g.nby) return;
  const int w = g.w, X0 = (tile % g.nbx) * TX, Y0 = (tile / g.nbx) * TY;
  // candidate ranges, exactly as in k_spread
  int o = X0 - (w - 1); o %= g.nx; if (o < 0) o += g.nx;
  const int len = min(TX, g.nx - X0) + w - 1;
  const int b0 = o / TX, b1 = (o + len - 1 < g.nx) ? (o + len - 1) / TX : g.nbx - 1;
  const int wrap_b1 = (o + len - 1 < g.nx) ? -1 : (o + len - 1 - g.nx) / TX;
  int bys[MAXB];
  const int ncy = origin_bins(Y0, min(TY, g.ny - Y0), TY, w, g.ny, bys);
  const int per_row = wrap_b1 >= 0 ? 2 : 1;
  const int nr = ncy * per_row;
  int beg = 0, cnt = 0;
  if (lane < nr) {
    const int row = bys[lane / per_row], piece = lane % per_row;
    const int ba = piece == 0 ? b0 : 0, bb = piece == 0 ? b1 : min(wrap_b1, b0 - 1);
    beg = bin_start[row * g.nbx + ba];
    cnt = bb >= ba ? bin_start[row * g.nbx + bb + 1] - beg : 0;
  }
  int incl = cnt;
#pragma unroll
  for (int o2 = 1; o2 < 16; o2 <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o2); if (lane >= o2) incl += v; }
  const int total = __shfl_sync(0xffffffffu, incl, MAXR - 1);
  const int excl = incl - cnt;
  const int TXe = min(TX, g.nx - X0), TYe = min(TY, g.ny - Y0);
  int nk = 0;
  for (int c0 = 0; c0 < total; c0 += 32) {
    const int c = c0 + lane;
    int r = 0;
#pragma unroll
    for (int q = 0; q < MAXR; ++q) { const int iq = __shfl_sync(0xffffffffu, incl, q); r += (c >= iq) ? 1 : 0; }
    r = r < MAXR ? r : MAXR - 1;
    const int rb = __shfl_sync(0xffffffffu, beg, r), re = __shfl_sync(0xffffffffu, excl, r);
    bool keep = false;
    int src = 0;
    if (c < total) {
      src = rb + (c - re);
      const int4 m = meta[src];
      int dx = X0 - m.x; if (dx < 0) dx += g.nx;
      int ex = m.x - X0; if (ex < 0) ex += g.nx;
      int dy = Y0 - m.y; if (dy < 0) dy += g.ny;
      int ey = m.y - Y0; if (ey < 0) ey += g.ny;
      keep = (m.z <= m.w) && (dx < w || ex < TXe) && (dy < w || ey < TYe);
    }
    const unsigned bal = __ballot_sync(0xffffffffu, keep);
    const int slot = nk + __popc(bal & ((1u << lane) - 1));
    if (keep && slot < LMAX) tile_list[(size_t)tile * LMAX + slot] = src;
    nk += __popc(bal);
  }
  if (lane == 0) {
    tile_cnt[tile] = nk;
    if (nk > pc_limit) ov_tiles[atomicAdd(ov_count, 1)] = tile;
  }
}

__device__ __forceinline__ void cp_async4(int* smem_dst, const int* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async16v(void* smem_dst, const void* gmem_src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}

// Persistent CTAs (DP_SPREAD_MINB per SM) walk the tiles b, b + G, ... with everything that comes from global memory two steps ahead:
// while tile k is accumulated from one staging buffer, the records, values and footprints of tile k + 1 arrive in the other one
// (cp.async) and the survivor list of tile k + 2 in a third small slot — one __syncthreads per tile, no global latency on the
// critical path.  Tiles whose list does not fit a chunk are skipped (k_spread takes them from the overflow list).
template <int NZ, class GT, int MODE>
__global__ void __launch_bounds__(SPREAD_THREADS, DP_SPREAD_MINB) k_spread_pipe(SpreadArgs A, const int* __restrict__ tile_cnt, const int* __restrict__ tile_list) {
  typedef SpreadBuf<NZ, MODE> SB;
  constexpr int NL = SB::NL, WREC = SB::WREC, WS = SB::WS, NREC = SB::NREC, PC = SB::PC, LS = LMAX + 1;
  extern __shared__ __align__(16) unsigned char spread_smem[];
  SB* B = reinterpret_cast<SB*>(spread_smem);                 // two staging buffers
  int* s_list = reinterpret_cast<int*>(B + 2);                // three list slots: LMAX indices + the count

  const GridGeom& g = A.g;
  const int grp = blockIdx.y, ntiles = g.nbx * g.nby, G = gridDim.x;
  const int t = threadIdx.x;
  const int ti = t % TX, tj = (t / TX) % TY, tz = t / (TX * TY);

  auto load_list = [&](int k, int tile) {
    if (tile >= ntiles) return;
    int* L = s_list + (k % 3) * LS;
    if (t < LMAX) cp_async4(L + t, tile_list + (size_t)tile * LMAX + t);
    else if (t == LMAX) cp_async4(L + LMAX, tile_cnt + tile);
  };
  auto stage = [&](int k, int tile) {
    if (tile >= ntiles) return;
    const int* L = s_list + (k % 3) * LS;
    const int nl = L[LMAX];
    if (nl > PC) return;
    SB& b = B[k & 1];
    if (t < nl) {
      const int p = L[t];
      cp_async16v(&b.meta[t], A.meta + p);
      if (MODE) {
#pragma unroll
        for (int c = 0; c < 3; ++c) { cp_async8(&b.val[t][c], A.val_s[0] + 3 * (size_t)p + c); cp_async8(&b.val[t][3 + c], A.val_s[1] + 3 * (size_t)p + c); }
      } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) cp_async8(&b.val[t][c], A.val_s[grp] + 3 * (size_t)p + c);
      }
    }
    if constexpr (WREC % 2 == 0) {
      constexpr int WH = WS / 2;
      for (int i = t; i < nl * NREC * WH; i += SPREAD_THREADS) {
        const int q = i / (NREC * WH), rem = i - q * (NREC * WH), k2 = rem / WH, e = 2 * (rem - k2 * WH);
        const int kk = MODE ? k2 : grp;
        if (e < WREC) cp_async16(&b.w[q][k2][e], A.wrec + ((size_t)kk * A.cap + L[q]) * WREC + e);
        else { b.w[q][k2][e] = 0.0; b.w[q][k2][e + 1] = 0.0; }
      }
    } else {
      for (int i = t; i < nl * NREC * WS; i += SPREAD_THREADS) {
        const int q = i / (NREC * WS), rem = i - q * (NREC * WS), k2 = rem / WS, e = rem - k2 * WS;
        const int kk = MODE ? k2 : grp;
        if (e < WREC) cp_async8(&b.w[q][k2][e], A.wrec + ((size_t)kk * A.cap + L[q]) * WREC + e);
        else b.w[q][k2][e] = 0.0;
      }
    }
  };

  const int tile0 = blockIdx.x;
  load_list(0, tile0);
  load_list(1, tile0 + G);
  cp_async_wait_all_groups();
  __syncthreads();
  stage(0, tile0);
  for (int k = 0, tile = tile0; tile < ntiles; ++k, tile += G) {
    cp_async_wait_all_groups();                               // records of tile k, list of tile k + 1
    __syncthreads();                                          // ... visible to all; every thread is done with tile k - 1
    load_list(k + 2, tile + 2 * G);
    stage(k + 1, tile + G);
    const int nl = s_list[(k % 3) * LS + LMAX];
    if (nl > PC) continue;                                    // overflow tile: left to k_spread
    const int X0 = (tile % g.nbx) * TX, Y0 = (tile / g.nbx) * TY;
    const int gi = X0 + ti, gj = Y0 + tj;
    const bool in_grid = gi < g.nx && gj < g.ny;
    GT acc[NL][3];
#pragma unroll
    for (int li = 0; li < NL; ++li) { acc[li][0] = 0; acc[li][1] = 0; acc[li][2] = 0; }
    accumulate_chunk<NZ, GT, MODE>(acc, B[k & 1], nl, g, gi, gj, tz, in_grid);
    store_tile<NZ, GT>(acc, A, g, grp, gi, gj, tz, in_grid);
  }
  cp_async_wait_all_groups();
}

// ---------------------------------------------------------------------------------------------- interpolate
struct InterpArgs {
  GridGeom g;
  const int* perm;
  const int4* meta;
  const double* wrec;
  size_t cap;
  const double* zweights;    // h^2 (H/2) w_l
  const double* grid;
  size_t real_field;
  double* U;
  double* Omega;             // may be NULL
};

#define DP_INTERP_WARPS 16
constexpr int INTERP_WARPS = DP_INTERP_WARPS;

// One warp per particle (sorted order, so neighbouring warps gather from neighbouring columns): the lanes sweep the
// w x w x (lmax-lmin+1) footprint, weights come from the particle's records, the six sums are reduced by shuffles.
// W = kernel support (compile-time: the footprint index arithmetic of the inner loop then has no integer division)
// MODE 0: U from fields 0-2 with Delta_M, Omega from fields 3-5 (= (1/2) curl u) with Delta_D   (eqs 10, 11);
// MODE 1 (kernel-derivative torques): U as before, Omega = (1/2) sum_g (u x G) h^2 (H/2) w_l from the SAME three fields.
#define DP_INTERP_MINB 1
template <class GT, int W, int MODE>
__global__ void __launch_bounds__(INTERP_WARPS * 32, DP_INTERP_MINB) k_interp(int n, InterpArgs A) {
  constexpr int NREC = MODE ? 3 : 2;
  // dynamic shared memory: quadrature weights [DP_MAX_NZ], then two sets of per-warp weight records [2][INTERP_WARPS][NREC][WR]: while a
  // warp gathers for one particle, the records (and the footprint record, in registers) of its next particle are already on their way
  extern __shared__ __align__(16) double interp_smem[];
  double* s_zw = interp_smem;
  const GridGeom& g = A.g;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  constexpr int w = W;
  const int nz = g.nz, wrec = 2 * DP_MAX_W + nz, WR = (wrec + 1) & ~1;
  double* s_wb = interp_smem + DP_MAX_NZ;
  for (int i = threadIdx.x; i < nz; i += blockDim.x) s_zw[i] = A.zweights[i];
  __syncthreads();
  const int nk = A.Omega ? NREC : 1;
  auto wbuf = [&](int b) { return s_wb + (size_t)((b * INTERP_WARPS + wid) * NREC) * WR; };
  auto prefetch = [&](int b, int pp) {
    double* d = wbuf(b);
    for (int k = 0; k < nk; ++k) {
      const double* rec = A.wrec + ((size_t)k * A.cap + pp) * wrec;
      for (int e = lane; e < wrec; e += 32) cp_async8(d + k * WR + e, rec + e);
    }
    cp_async_commit_only();
  };
  const int stride = gridDim.x * INTERP_WARPS;
  int p = blockIdx.x * INTERP_WARPS + wid, cur = 0;
  int4 m = make_int4(0, 0, 1, 0);
  int dst = 0;
  if (p < n) { m = A.meta[p]; dst = A.perm[p]; prefetch(0, p); }
  for (; p < n; p += stride) {
    const int pn = p + stride;
    int4 mn = make_int4(0, 0, 1, 0);
    int dstn = 0;
    if (pn < n) { mn = A.meta[pn]; dstn = A.perm[pn]; }
    cp_async_wait_only();
    __syncwarp();                                  // this particle's records are in buffer cur; every lane is done with the other buffer
    if (pn < n) prefetch(cur ^ 1, pn);
    const double* swb = wbuf(cur);
    GT s[6] = {0, 0, 0, 0, 0, 0};
    if (m.z <= m.w) {
      constexpr int ww = w * w;
      const int nent = (m.w - m.z + 1) * ww;
#pragma unroll 4
      for (int e = lane; e < nent; e += 32) {
        int l = m.z + e / ww, rem = e % ww, b = rem / w, a = rem % w;
        int i = m.x + a; if (i >= g.nx) i -= g.nx;
        int j = m.y + b; if (j >= g.ny) j -= g.ny;
        const size_t off = ((size_t)l * g.ny + j) * g.nx + i;
        const GT wl = (GT)s_zw[l];
        if (MODE == 0) {
          for (int k = 0; k < nk; ++k) {
            const double* sw = swb + k * WR;
            const GT wgt = (GT)sw[a] * (GT)sw[DP_MAX_W + b] * (GT)sw[2 * DP_MAX_W + l];
            const GT* gp = reinterpret_cast<const GT*>(A.grid) + (size_t)(3 * k) * A.real_field + off;
            s[3 * k + 0] += __ldg(gp) * wgt * wl;
            s[3 * k + 1] += __ldg(gp + A.real_field) * wgt * wl;
            s[3 * k + 2] += __ldg(gp + 2 * A.real_field) * wgt * wl;
          }
        } else {
          const GT* gp = reinterpret_cast<const GT*>(A.grid) + off;
          const GT u = __ldg(gp) * wl, v = __ldg(gp + A.real_field) * wl, ww2 = __ldg(gp + 2 * A.real_field) * wl;
          const double* wM = swb;
          const GT wgt = (GT)wM[a] * (GT)wM[DP_MAX_W + b] * (GT)wM[2 * DP_MAX_W + l];
          s[0] += u * wgt; s[1] += v * wgt; s[2] += ww2 * wgt;
          if (nk > 1) {
            const double* wD = swb + (MODE ? 1 : 0) * WR; const double* wG = swb + (MODE ? 2 : 0) * WR;
            const GT zD = (GT)wD[2 * DP_MAX_W + l];
            const GT Gx = (GT)wG[a] * (GT)wD[DP_MAX_W + b] * zD, Gy = (GT)wD[a] * (GT)wG[DP_MAX_W + b] * zD;
            const GT Gz = (GT)wD[a] * (GT)wD[DP_MAX_W + b] * (GT)wG[2 * DP_MAX_W + l];
            s[3] += (GT)0.5 * (v * Gz - ww2 * Gy);                       // (1/2) (u x G)
            s[4] += (GT)0.5 * (ww2 * Gx - u * Gz);
            s[5] += (GT)0.5 * (u * Gy - v * Gx);
          }
        }
      }
    }
    const int nsum = A.Omega ? 6 : 3;
    for (int c = 0; c < nsum; ++c)
      for (int o = 16; o > 0; o >>= 1) s[c] += __shfl_xor_sync(0xffffffffu, s[c], o);
    if (lane < 3) A.U[3 * (size_t)dst + lane] = (double)(lane == 0 ? s[0] : (lane == 1 ? s[1] : s[2]));
    if (A.Omega && lane >= 3 && lane < 6) A.Omega[3 * (size_t)dst + lane - 3] = (double)(lane == 3 ? s[3] : (lane == 4 ? s[4] : s[5]));
    m = mn; dst = dstn; cur ^= 1;
  }
}

GridGeom make_geom(const dp_plan* P) {
  GridGeom g;
  g.nx = P->p.nx; g.ny = P->p.ny; g.nz = P->p.nz; g.w = P->p.w; g.wall_mode = P->p.wall_mode;
  g.nbx = P->nbx; g.nby = P->nby;
  g.Lx = P->p.Lx; g.Ly = P->p.Ly; g.H = P->p.H; g.h = P->h; g.alpha = P->alpha;
  return g;
}

}  // namespace

cudaError_t dp_launch_bin(dp_plan* P, int n, const double* pos, const double* force, const double* torque, bool dense, cudaStream_t st) {
  GridGeom g = make_geom(P);
  cudaError_t e = cudaMemsetAsync(P->d_bin_count, 0, sizeof(int) * P->nbins, st);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(P->d_lmin, 0x7f, sizeof(int), st);          // 0x7f7f7f7f: "no plane touched yet"
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(P->d_flag, 0, sizeof(int), st);
  if (e != cudaSuccess) return e;
  const int T = 256, B = (n + T - 1) / T;
  k_bin_count<<<B, T, 0, st>>>(n, pos, g, P->d_bin_of, P->d_slot_of, P->d_bin_count, P->d_flag);
  const int nsb = (P->nbins + SCAN_CHUNK - 1) / SCAN_CHUNK;      // P->d_scan_sums holds nsb ints (plan.cu)
  k_scan_local<<<nsb, SCAN_THREADS, 0, st>>>(P->nbins, P->d_bin_count, P->d_bin_start, P->d_scan_sums);
  k_scan_add<<<nsb, SCAN_THREADS, 0, st>>>(P->nbins, nsb, P->d_bin_start, P->d_scan_sums);
  k_bin_scatter<<<B, T, 0, st>>>(n, pos, force, torque, g, P->d_bin_of, P->d_slot_of, P->d_bin_start, P->d_znodes, P->d_perm, P->d_meta,
                                P->d_pos_s, P->d_frc_s, P->torques ? P->d_trq_s : nullptr, P->d_lmin);
  if (dense) { e = cudaMemsetAsync(P->d_lmin, 0, sizeof(int), st); if (e != cudaSuccess) return e; }   // every plane is transformed
  return cudaGetLastError();
}

// setup_only: set the kernel attributes of the plan's spread kernels and return (called once per plan from dp_create, never per product)
static cudaError_t spread_dispatch(dp_plan* P, int n, bool with_torque, cudaStream_t st, bool setup_only);
cudaError_t dp_launch_spread(dp_plan* P, int n, bool with_force, bool with_torque, cudaStream_t st) {
  (void)with_force;
  return spread_dispatch(P, n, with_torque, st, false);
}
static cudaError_t spread_dispatch(dp_plan* P, int n, bool with_torque, cudaStream_t st, bool setup_only) {
  const bool kt = P->kernel_torque;
  const int ngroups = (with_torque && !kt) ? 2 : 1;
  {
    // weight records of every envelope of the plan (the dipole records are also needed when only Omega is wanted)
    WeightArgs W;
    W.g = make_geom(P);
    W.pos_s = P->d_pos_s; W.meta = P->d_meta; W.znodes = P->d_znodes;
    W.beta[0] = P->p.beta_M; W.beta[1] = P->p.beta_D; W.beta[2] = P->p.beta_D;
    W.inv_Z[0] = 1.0 / P->ZM; W.inv_Z[1] = 1.0 / P->ZD; W.inv_Z[2] = 1.0 / P->ZD; W.inv_alpha = 1.0 / P->alpha;
    W.ucut = P->ucutD;
    W.wrec = P->d_wrec; W.cap = (size_t)P->p.max_particles;
    if (n > 0 && !setup_only) k_weights<<<(unsigned)((n + WEIGHT_WARPS - 1) / WEIGHT_WARPS), WEIGHT_WARPS * 32, 0, st>>>(n, W, P->nrec);
  }
  SpreadArgs A;
  A.g = make_geom(P);
  A.val_s[0] = P->d_frc_s; A.val_s[1] = P->d_trq_s;
  A.field0[0] = 0; A.field0[1] = 3;
  A.bin_start = P->d_bin_start;
  A.meta = P->d_meta;
  A.wrec = P->d_wrec; A.cap = (size_t)P->p.max_particles;
  A.grid = P->d_real;
  A.real_field = P->real_field;
  A.lmin = P->d_lmin;
  const bool f32 = P->p.transfer_fp32 != 0;
  // survivor lists per tile, then the pipelined kernel over the tiles whose list fits a staged chunk, then the culling kernel over the rest
  const int ntiles = P->nbx * P->nby;
  const int pc_limit = kt ? PCH / 2 : PCH;
  cudaError_t e = cudaSuccess;
  if (!setup_only) {
  e = cudaMemsetAsync(P->d_ov_count, 0, sizeof(int), st);
  if (e != cudaSuccess) return e;
  k_tile_lists<<<(ntiles + LIST_WARPS - 1) / LIST_WARPS, LIST_WARPS * 32, 0, st>>>(A.g, P->d_bin_start, P->d_meta, pc_limit, P->d_tile_cnt, P->d_tile_list,
                                                                                    P->d_ov_tiles, P->d_ov_count);
  }
  const int sms = P->sm_count;
#define DP_SPREAD_LAUNCH(NZV, GT, MODE)                                                                                                   \
  {                                                                                                                                      \
    constexpr int NZ = NZV;                                                                                                              \
    const int per_sm = DP_SPREAD_MINB;                                                                                                   \
    const size_t smem = 2 * sizeof(SpreadBuf<NZ, MODE>) + 3 * (LMAX + 1) * sizeof(int);                                                  \
    if (setup_only) return cudaFuncSetAttribute(k_spread_pipe<NZ, GT, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);    \
    const int gp = ntiles < sms * per_sm ? ntiles : sms * per_sm;                                                                        \
    k_spread_pipe<NZ, GT, MODE><<<dim3(gp, ngroups), SPREAD_THREADS, smem, st>>>(A, P->d_tile_cnt, P->d_tile_list);                      \
    k_spread<NZ, GT, MODE><<<dim3(gp, 1, ngroups), SPREAD_THREADS, 0, st>>>(A, P->d_ov_tiles, P->d_ov_count);                            \
  }
#define DP_SPREAD_CASE(NZ)                                                                        \
  case NZ:                                                                                        \
    if (kt) { if (f32) DP_SPREAD_LAUNCH(NZ, float, 1) else DP_SPREAD_LAUNCH(NZ, double, 1) }      \
    else    { if (f32) DP_SPREAD_LAUNCH(NZ, float, 0) else DP_SPREAD_LAUNCH(NZ, double, 0) }      \
    break;
  switch (P->p.nz) {
    DP_SPREAD_CASE(16) DP_SPREAD_CASE(19) DP_SPREAD_CASE(24) DP_SPREAD_CASE(26) DP_SPREAD_CASE(32) DP_SPREAD_CASE(40) DP_SPREAD_CASE(48) DP_SPREAD_CASE(64)
    default: return cudaErrorInvalidValue;
  }
#undef DP_SPREAD_CASE
#undef DP_SPREAD_LAUNCH
  return cudaGetLastError();
}

static cudaError_t interp_dispatch(dp_plan* P, int n, double* U, double* Omega, cudaStream_t st, bool setup_only);
cudaError_t dp_launch_interp(dp_plan* P, int n, double* U, double* Omega, cudaStream_t st) { return interp_dispatch(P, n, U, Omega, st, false); }
// once per plan, from dp_create: dynamic shared-memory limits of the plan's spread and interpolation kernels.  The interpolation kernel's size
// depends on nz while its instantiation does not, and the limit belongs to the function (not the plan): it is raised to the device's opt-in
// maximum so that plans with different nz can coexist.
cudaError_t dp_transfer_setup(dp_plan* P) {
  cudaError_t e = spread_dispatch(P, 0, false, nullptr, true);
  if (e != cudaSuccess) return e;
  return interp_dispatch(P, 0, nullptr, nullptr, nullptr, true);
}
static cudaError_t interp_dispatch(dp_plan* P, int n, double* U, double* Omega, cudaStream_t st, bool setup_only) {
  InterpArgs A;
  A.g = make_geom(P);
  A.perm = P->d_perm; A.meta = P->d_meta;
  A.wrec = P->d_wrec; A.cap = (size_t)P->p.max_particles;
  A.zweights = P->d_zweights;
  A.grid = P->d_real; A.real_field = P->real_field;
  A.U = U; A.Omega = Omega;
  int blocks = (n + INTERP_WARPS - 1) / INTERP_WARPS;
#define DP_INTERP_MAXB 32
  const int maxb = P->sm_count * DP_INTERP_MAXB;
  if (blocks > maxb) blocks = maxb;
  if (blocks < 1) blocks = 1;
  const bool f32 = P->p.transfer_fp32 != 0, kt = P->kernel_torque;
  const int wr_even = (2 * DP_MAX_W + P->p.nz + 1) & ~1;
  const size_t ismem = sizeof(double) * (DP_MAX_NZ + (size_t)2 * INTERP_WARPS * (kt ? 3 : 2) * wr_even);
#define DP_INTERP_LAUNCH(GT, WW, MODE)                                                                                           \
  { if (setup_only) return cudaFuncSetAttribute(k_interp<GT, WW, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, P->smem_optin); \
    k_interp<GT, WW, MODE><<<blocks, INTERP_WARPS * 32, ismem, st>>>(n, A); }
#define DP_INTERP_CASE(WW)                                                              \
  case WW:                                                                              \
    if (kt) { if (f32) DP_INTERP_LAUNCH(float, WW, 1) else DP_INTERP_LAUNCH(double, WW, 1) } \
    else    { if (f32) DP_INTERP_LAUNCH(float, WW, 0) else DP_INTERP_LAUNCH(double, WW, 0) } \
    break;
  switch (P->p.w) {
    DP_INTERP_CASE(4) DP_INTERP_CASE(5) DP_INTERP_CASE(6) DP_INTERP_CASE(7) DP_INTERP_CASE(8)
    default: return cudaErrorInvalidValue;
  }
#undef DP_INTERP_CASE
#undef DP_INTERP_LAUNCH
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------- binning with no allocation (dp_bin_particles_static)
#include <mutex>
// Step a0 for callers that must not allocate device memory: code running inside a framework that reserved all of HBM for its own pool at start-up,
// a plug-in whose host forbids driver allocations after initialisation (each one may synchronise the device, and the hot loop must not stall or
// fail with "out of memory" half way), or a worker that only ever gets buffers handed to it.  The product path keeps the work arrays of its
// counting sort in the plan (cudaMalloc in dp_create); here the same kernels run on a fixed array that is part of the loaded library image.
namespace {

static_assert(DP_BIN_TILE_X == TX && DP_BIN_TILE_Y == TY, "dp.h states the tile of the sort");
constexpr int SB_MAX_N = DP_STATIC_BIN_MAX_PARTICLES, SB_MAX_BINS = DP_STATIC_BIN_MAX_TILES;
constexpr int SB_SCAN = SB_MAX_BINS / SCAN_CHUNK + 1;
// layout (ints): tile of each particle [SB_MAX_N] | rank within its tile [SB_MAX_N] | tile counters [SB_MAX_BINS] | chunk totals of the scan [SB_SCAN] | flag [1]
constexpr size_t SB_OFF_SLOT = SB_MAX_N, SB_OFF_COUNT = 2 * (size_t)SB_MAX_N, SB_OFF_SUMS = SB_OFF_COUNT + SB_MAX_BINS, SB_OFF_FLAG = SB_OFF_SUMS + SB_SCAN;
constexpr size_t SB_INTS = SB_OFF_FLAG + 1;
// 2.5 MiB that every GPU which loads libdpstokes.so holds until the process exits.  In host code this name is only a handle for
// cudaGetSymbolAddress — it is NOT a device address and must never be passed to a kernel as it stands.
static __device__ __align__(256) int g_static_bin_scratch[SB_INTS];

constexpr int SB_MAX_DEVICES = 64;
std::mutex g_sb_mutex;
int* g_sb_addr[SB_MAX_DEVICES] = {};            // device address of g_static_bin_scratch on each device, resolved once per device

// `dev` must be the current device: the symbol is looked up in the current device's copy of the module
cudaError_t static_bin_scratch(int dev, int** out) {
  std::lock_guard<std::mutex> lock(g_sb_mutex);
  if (!g_sb_addr[dev]) {
    void* a = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&a, g_static_bin_scratch);
    if (e != cudaSuccess) return e;
    g_sb_addr[dev] = static_cast<int*>(a);
  }
  *out = g_sb_addr[dev];
  return cudaSuccess;
}

// the part of k_bin_scatter that a caller of the sort alone needs: sorted slot -> original particle index
__global__ void k_bin_perm(int n, const int* __restrict__ bin_of, const int* __restrict__ slot_of, const int* __restrict__ bin_start, int* __restrict__ perm) {
  const int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p < n) perm[bin_start[bin_of[p]] + slot_of[p]] = p;
}

}  // namespace

extern "C" int dp_bin_particles_static(const dp_params* prm, int n, const double* pos, int* perm, int* tile_start, void* cuda_stream) {
  if (!prm || !tile_start || n < 0 || (n > 0 && (!pos || !perm))) return DP_EINVAL;
  const dp_params& p = *prm;
  // the geometry checks of dp_create that binning depends on
  if (p.wall_mode != DP_BOTTOM_WALL && p.wall_mode != DP_SLIT) return DP_EINVAL;
  if (!(p.Lx > 0) || !(p.Ly > 0) || !(p.H > 0) || p.w < 4 || p.w > DP_MAX_W) return DP_EINVAL;
  if (p.nx < TX + p.w || p.ny < TY + p.w || (p.nx & 1) || (p.ny & 1)) return DP_EINVAL;
  const double h = p.Lx / p.nx;
  if (fabs(h - p.Ly / p.ny) > 1e-12 * h) return DP_EINVAL;
  if (p.device < 0 || p.device >= SB_MAX_DEVICES) return DP_EINVAL;
  GridGeom g;
  g.nx = p.nx; g.ny = p.ny; g.nz = p.nz; g.w = p.w; g.wall_mode = p.wall_mode;
  g.nbx = (p.nx + TX - 1) / TX; g.nby = (p.ny + TY - 1) / TY;
  g.Lx = p.Lx; g.Ly = p.Ly; g.H = p.H; g.h = h; g.alpha = 0.5 * p.w * h;
  const long long nbins_ll = (long long)g.nbx * g.nby;
  if (n > SB_MAX_N || nbins_ll > SB_MAX_BINS) return DP_ETOOBIG;      // beyond the fixed work array: use a plan (dp_create) instead
  const int nbins = (int)nbins_ll;

  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return DP_ECUDA; }
  if (prev != p.device && cudaSetDevice(p.device) != cudaSuccess) { cudaGetLastError(); return DP_ECUDA; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int* S = nullptr;
  cudaError_t e = static_bin_scratch(p.device, &S);
  // The array still holds what the previous call left in it: the tile counters and the flag are the two parts that must start at zero
  // (everything else is written before it is read).  A memset on the stream allocates nothing.
  if (e == cudaSuccess) e = cudaMemsetAsync(S + SB_OFF_COUNT, 0, sizeof(int) * (size_t)nbins, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(S + SB_OFF_FLAG, 0, sizeof(int), st);
  if (e == cudaSuccess) {
    const int T = 256, B = (n + T - 1) / T;
    if (n > 0) k_bin_count<<<B, T, 0, st>>>(n, pos, g, S, S + SB_OFF_SLOT, S + SB_OFF_COUNT, S + SB_OFF_FLAG);
    const int nsb = (nbins + SCAN_CHUNK - 1) / SCAN_CHUNK;
    k_scan_local<<<nsb, SCAN_THREADS, 0, st>>>(nbins, S + SB_OFF_COUNT, tile_start, S + SB_OFF_SUMS);
    k_scan_add<<<nsb, SCAN_THREADS, 0, st>>>(nbins, nsb, tile_start, S + SB_OFF_SUMS);
    if (n > 0) k_bin_perm<<<B, T, 0, st>>>(n, S, S + SB_OFF_SLOT, tile_start, perm);
    e = cudaGetLastError();
  }
  if (prev != p.device) cudaSetDevice(prev);
  if (e != cudaSuccess) { cudaGetLastError(); return DP_ECUDA; }
  return DP_OK;
}
