// transfer.cu — particle <-> grid kernels: binning (a0), spreading (a1, a2; paper step 1), interpolation (a12; step 8).
//
// Step 1 (eqs 7, 9, 53, 54): f(x_g) = sum_j F_j Delta_M^W(x_g - r_j), t(x_g) = sum_j tau_j Delta_D^W(x_g - r_j)
//   Delta^W = phi(x)phi(y)[phi(z - z_j) - phi(z + z_j) - (slit) phi(z - (2H - z_j))]
// Step 8 (eqs 10, 11): U_j = sum_g u(x_g) Delta_M^W(x_g - r_j) h^2 (H/2) w_l, Omega_j likewise with Delta_D^W.
//
// B200 design: particles are counting-sorted by the xy tile (16 x 8 grid columns) that contains the origin of
// their w x w footprint.  One CTA owns one tile of one field triple: it accumulates every footprint that touches
// the tile into a shared-memory tile [3][nz][8][16] (each thread owns one column and a fixed residue class of the plane index, so no
// atomics and no conflicts), then streams the whole tile to HBM once with 16-byte coalesced stores — every grid
// value is written exactly once, zeros included, so there is no memset pass and no global atomic.
#include "common.cuh"

namespace {

constexpr int TX = DP_TILE_X, TY = DP_TILE_Y;
constexpr int ZSPLIT = 2;                       // z residue classes per column
constexpr int SPREAD_THREADS = TX * TY * ZSPLIT;
constexpr int PCH = 16;                         // particles staged per chunk

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
  while (left > 0 && cnt < 4) {
    int b = o / T, bend = min((b + 1) * T, n);
    out[cnt++] = b;
    left -= bend - o;
    o = bend == n ? 0 : bend;
  }
  return cnt;
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

// exclusive scan of bin_count -> bin_start[0..nbins]; one CTA, chunked
__global__ void k_scan(int nbins, const int* __restrict__ cnt, int* __restrict__ start) {
  __shared__ int warp_sums[32];
  __shared__ int carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int base = 0; base < nbins; base += blockDim.x) {
    int i = base + threadIdx.x;
    int v = i < nbins ? cnt[i] : 0;
    int s = v;
    for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += t; }
    if (lane == 31) warp_sums[wid] = s;
    __syncthreads();
    if (wid == 0) {
      int ws = lane < nw ? warp_sums[lane] : 0;
      for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, ws, o); if (lane >= o) ws += t; }
      warp_sums[lane] = ws;
    }
    __syncthreads();
    int excl = carry + (wid > 0 ? warp_sums[wid - 1] : 0) + s - v;
    if (i < nbins) start[i] = excl;
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) carry = excl + v;
    __syncthreads();
  }
  if (threadIdx.x == 0) start[nbins] = carry;
}

__global__ void k_bin_scatter(int n, const double* __restrict__ pos, const double* __restrict__ force,
                              const double* __restrict__ torque, GridGeom g, const int* __restrict__ bin_of,
                              const int* __restrict__ slot_of, const int* __restrict__ bin_start, int* __restrict__ perm,
                              double* __restrict__ pos_s, double* __restrict__ frc_s, double* __restrict__ trq_s) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  int d = bin_start[bin_of[p]] + slot_of[p];
  perm[d] = p;
  double x = pos[3 * (size_t)p], y = pos[3 * (size_t)p + 1], z = pos[3 * (size_t)p + 2];
  bool ok = (z >= 0.0) && (z <= g.H) && (g.wall_mode == DP_SLIT || z + g.alpha <= g.H) && isfinite(x) && isfinite(y);
  double xw = 0.0, yw = 0.0;
  if (ok) { xw = x - floor(x / g.Lx) * g.Lx; yw = y - floor(y / g.Ly) * g.Ly; }
  pos_s[3 * (size_t)d] = xw; pos_s[3 * (size_t)d + 1] = yw; pos_s[3 * (size_t)d + 2] = ok ? z : -1.0;   // z < 0: skipped
  for (int c = 0; c < 3; ++c) {
    if (frc_s) frc_s[3 * (size_t)d + c] = force ? force[3 * (size_t)p + c] : 0.0;
    if (trq_s) trq_s[3 * (size_t)d + c] = torque ? torque[3 * (size_t)p + c] : 0.0;
  }
}

// ---------------------------------------------------------------------------------------------- z weights
// zeta(l; z_p) = phi(z_l - z_p) - phi(z_l + z_p) - [slit] phi(z_l - (2H - z_p))   (eq 9)
__device__ __forceinline__ double zeta_weight(double zl, double zp, double H, int wall_mode, double alpha, double beta, double Z) {
  double q, r, v = 0.0;
  q = (zl - zp) / alpha; if (fabs(q) <= 1.0) { r = 1.0 - q * q; r = r < 0.0 ? 0.0 : r; v += exp(beta * (sqrt(r) - 1.0)) / Z; }
  q = (zl + zp) / alpha; if (fabs(q) <= 1.0) { r = 1.0 - q * q; r = r < 0.0 ? 0.0 : r; v -= exp(beta * (sqrt(r) - 1.0)) / Z; }
  if (wall_mode == DP_SLIT) { q = (zl - (2.0 * H - zp)) / alpha; if (fabs(q) <= 1.0) { r = 1.0 - q * q; r = r < 0.0 ? 0.0 : r; v -= exp(beta * (sqrt(r) - 1.0)) / Z; } }
  return v;
}
__device__ __forceinline__ double xy_weight(double s, double alpha, double beta, double Z) {
  double q = s / alpha;
  if (!(fabs(q) <= 1.0)) return 0.0;
  double r = 1.0 - q * q; r = r < 0.0 ? 0.0 : r;
  return exp(beta * (sqrt(r) - 1.0)) / Z;
}
// node range with z_l in [max(0, zp - alpha), min(H, zp + alpha)] (nodes decrease with l); covers every image term
__device__ __forceinline__ void z_range(const double* zn, int nz, double zp, double alpha, double H, int& lmin, int& lmax) {
  double hi = zp + alpha, lo = zp - alpha;
  int a = 0, b = nz - 1;
  while (a < nz && zn[a] > hi) ++a;
  while (b >= 0 && zn[b] < lo) --b;
  lmin = a; lmax = b;
}

// ---------------------------------------------------------------------------------------------- spread
struct SpreadArgs {
  GridGeom g;
  const double* pos_s;
  const double* val_s[2];    // forces, torques (sorted)
  double beta[2], Z[2];
  int field0[2];             // first output field of each group
  int ngroups;
  const int* bin_start;
  const double* znodes;
  double* grid;
  size_t real_field;
};

__global__ void __launch_bounds__(SPREAD_THREADS) k_spread(SpreadArgs A) {
  extern __shared__ double smem[];
  const GridGeom& g = A.g;
  const int nz = g.nz, w = g.w;
  double* acc = smem;                                   // [3][nz][TY][TX]
  double* s_zn = acc + 3 * nz * TY * TX;                // [nz]
  double* s_wx = s_zn + nz;                             // [PCH][DP_MAX_W]
  double* s_wy = s_wx + PCH * DP_MAX_W;                 // [PCH][DP_MAX_W]
  double* s_zt = s_wy + PCH * DP_MAX_W;                 // [PCH][nz]
  double* s_val = s_zt + PCH * nz;                      // [PCH][3]
  int* s_meta = (int*)(s_val + PCH * 3);                // [PCH][4]: i0, j0, lmin, lmax

  const int grp = blockIdx.y;
  const int bx = blockIdx.x % g.nbx, by = blockIdx.x / g.nbx;
  const int X0 = bx * TX, Y0 = by * TY;
  const int t = threadIdx.x;
  const int ti = t % TX, tj = (t / TX) % TY, tz = t / (TX * TY);
  const int gi = X0 + ti, gj = Y0 + tj;
  const double beta = A.beta[grp], Z = A.Z[grp];
  const double* __restrict__ val = A.val_s[grp];

  for (int i = t; i < 3 * nz * TY * TX; i += SPREAD_THREADS) acc[i] = 0.0;
  for (int i = t; i < nz; i += SPREAD_THREADS) s_zn[i] = A.znodes[i];

  // origin bins whose footprints can reach this tile: origin columns in the cyclic range [X0-w+1, X0+TXeff-1]
  int bxs[4], bys[4];
  const int ncx = origin_bins(X0, min(TX, g.nx - X0), TX, w, g.nx, bxs);
  const int ncy = origin_bins(Y0, min(TY, g.ny - Y0), TY, w, g.ny, bys);

  for (int cy = 0; cy < ncy; ++cy) {
    for (int cx = 0; cx < ncx; ++cx) {
      const int b = bys[cy] * g.nbx + bxs[cx];
      const int pbeg = A.bin_start[b], pend = A.bin_start[b + 1];
      for (int c0 = pbeg; c0 < pend; c0 += PCH) {
        const int np = min(PCH, pend - c0);
        __syncthreads();
        // ---- phase A: footprint weights of the chunk
        if (t < np) {
          const double* r = A.pos_s + 3 * (size_t)(c0 + t);
          double zp = r[2];
          int lmin = 1, lmax = 0;
          int i0 = 0, j0 = 0;
          if (zp >= 0.0) {
            i0 = origin_cell(r[0], g.alpha, g.h, g.nx);
            j0 = origin_cell(r[1], g.alpha, g.h, g.ny);
            z_range(s_zn, nz, zp, g.alpha, g.H, lmin, lmax);
          }
          s_meta[4 * t] = i0; s_meta[4 * t + 1] = j0; s_meta[4 * t + 2] = lmin; s_meta[4 * t + 3] = lmax;
          for (int c = 0; c < 3; ++c) s_val[3 * t + c] = val[3 * (size_t)(c0 + t) + c];
        }
        for (int i = t; i < np * 2 * w; i += SPREAD_THREADS) {
          int q = i / (2 * w), rr = i % (2 * w);
          const double* r = A.pos_s + 3 * (size_t)(c0 + q);
          if (rr < w) {
            double xw = r[0];
            double i0 = ceil((xw - g.alpha) / g.h);         // unwrapped origin: distances use the unwrapped node
            s_wx[q * DP_MAX_W + rr] = xy_weight((i0 + rr) * g.h - xw, g.alpha, beta, Z);
          } else {
            double yw = r[1];
            double j0 = ceil((yw - g.alpha) / g.h);
            s_wy[q * DP_MAX_W + rr - w] = xy_weight((j0 + (rr - w)) * g.h - yw, g.alpha, beta, Z);
          }
        }
        for (int i = t; i < np * nz; i += SPREAD_THREADS) {
          int q = i / nz, l = i % nz;
          double zp = A.pos_s[3 * (size_t)(c0 + q) + 2];
          s_zt[q * nz + l] = zp >= 0.0 ? zeta_weight(s_zn[l], zp, g.H, g.wall_mode, g.alpha, beta, Z) : 0.0;
        }
        __syncthreads();
        // ---- phase B: each thread adds to its own column (ti, tj), z residue class tz
        for (int q = 0; q < np; ++q) {
          int a = gi - s_meta[4 * q]; if (a < 0) a += g.nx;
          int bb = gj - s_meta[4 * q + 1]; if (bb < 0) bb += g.ny;
          if (a < w && bb < w && gi < g.nx && gj < g.ny) {
            const double wxy = s_wx[q * DP_MAX_W + a] * s_wy[q * DP_MAX_W + bb];
            const double v0 = s_val[3 * q], v1 = s_val[3 * q + 1], v2 = s_val[3 * q + 2];
            const int lmin = s_meta[4 * q + 2], lmax = s_meta[4 * q + 3];
            // a thread owns the planes l = tz (mod ZSPLIT) of its column for EVERY particle: no two threads ever touch the same cell
            for (int l = lmin + ((tz - lmin) & (ZSPLIT - 1)); l <= lmax; l += ZSPLIT) {
              const double wgt = wxy * s_zt[q * nz + l];
              double* o = acc + (l * TY + tj) * TX + ti;
              o[0] += v0 * wgt;
              o[nz * TY * TX] += v1 * wgt;
              o[2 * nz * TY * TX] += v2 * wgt;
            }
          }
        }
      }
    }
  }
  __syncthreads();
  // ---- flush the tile: every value written once, 16-byte stores
  const int rows = 3 * nz * TY;
  for (int i = t; i < rows * (TX / 2); i += SPREAD_THREADS) {
    int row = i / (TX / 2), i2 = (i % (TX / 2)) * 2;
    int j = row % TY, l = (row / TY) % nz, c = row / (TY * nz);
    int col = X0 + i2, rowg = Y0 + j;
    if (col < g.nx && rowg < g.ny) {
      double2 v = *reinterpret_cast<const double2*>(acc + ((c * nz + l) * TY + j) * TX + i2);
      double* dst = A.grid + (size_t)(A.field0[grp] + c) * A.real_field + ((size_t)l * g.ny + rowg) * g.nx + col;
      *reinterpret_cast<double2*>(dst) = v;       // nx even, col even: 16-byte aligned
    }
  }
}

// ---------------------------------------------------------------------------------------------- interpolate
struct InterpArgs {
  GridGeom g;
  const double* pos_s;
  const int* perm;
  double beta[2], Z[2];
  const double* znodes;
  const double* zweights;    // h^2 (H/2) w_l
  const double* grid;
  size_t real_field;
  double* U;
  double* Omega;             // may be NULL
};

constexpr int INTERP_WARPS = 8;

__global__ void __launch_bounds__(INTERP_WARPS * 32) k_interp(int n, InterpArgs A) {
  __shared__ double s_w[INTERP_WARPS][2][2 * DP_MAX_W + DP_MAX_NZ];   // per warp, per kernel: wx[8], wy[8], zeta[nz]
  __shared__ double s_zn[DP_MAX_NZ], s_zw[DP_MAX_NZ];
  const GridGeom& g = A.g;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int nz = g.nz, w = g.w;
  for (int i = threadIdx.x; i < nz; i += blockDim.x) { s_zn[i] = A.znodes[i]; s_zw[i] = A.zweights[i]; }
  __syncthreads();
  const int nk = A.Omega ? 2 : 1;
  for (int p = blockIdx.x * INTERP_WARPS + wid; p < n; p += gridDim.x * INTERP_WARPS) {
    const double xw = A.pos_s[3 * (size_t)p], yw = A.pos_s[3 * (size_t)p + 1], zp = A.pos_s[3 * (size_t)p + 2];
    const int dst = A.perm[p];
    double s[6] = {0, 0, 0, 0, 0, 0};
    if (zp >= 0.0) {
      const double fi0 = ceil((xw - g.alpha) / g.h), fj0 = ceil((yw - g.alpha) / g.h);
      int i0 = (int)fi0 % g.nx; if (i0 < 0) i0 += g.nx;
      int j0 = (int)fj0 % g.ny; if (j0 < 0) j0 += g.ny;
      int lmin, lmax;
      z_range(s_zn, nz, zp, g.alpha, g.H, lmin, lmax);
      __syncwarp();
      for (int k = 0; k < nk; ++k) {
        double* sw = s_w[wid][k];
        if (lane < w) sw[lane] = xy_weight((fi0 + lane) * g.h - xw, g.alpha, A.beta[k], A.Z[k]);
        else if (lane >= 8 && lane < 8 + w) sw[DP_MAX_W + lane - 8] = xy_weight((fj0 + (lane - 8)) * g.h - yw, g.alpha, A.beta[k], A.Z[k]);
        for (int l = lmin + lane; l <= lmax; l += 32)
          sw[2 * DP_MAX_W + l] = zeta_weight(s_zn[l], zp, g.H, g.wall_mode, g.alpha, A.beta[k], A.Z[k]);
      }
      __syncwarp();
      const int ww = w * w, nent = (lmax - lmin + 1) * ww;
      for (int e = lane; e < nent; e += 32) {
        int l = lmin + e / ww, rem = e % ww, b = rem / w, a = rem % w;
        int i = i0 + a; if (i >= g.nx) i -= g.nx;
        int j = j0 + b; if (j >= g.ny) j -= g.ny;
        const size_t off = ((size_t)l * g.ny + j) * g.nx + i;
        const double wl = s_zw[l];
        for (int k = 0; k < nk; ++k) {
          const double* sw = s_w[wid][k];
          const double wgt = sw[a] * sw[DP_MAX_W + b] * sw[2 * DP_MAX_W + l];
          const double* gp = A.grid + (size_t)(3 * k) * A.real_field + off;
          s[3 * k + 0] += __ldg(gp) * wgt * wl;
          s[3 * k + 1] += __ldg(gp + A.real_field) * wgt * wl;
          s[3 * k + 2] += __ldg(gp + 2 * A.real_field) * wgt * wl;
        }
      }
    }
    for (int c = 0; c < 3 * nk; ++c)
      for (int o = 16; o > 0; o >>= 1) s[c] += __shfl_xor_sync(0xffffffffu, s[c], o);
    if (lane < 3) A.U[3 * (size_t)dst + lane] = lane == 0 ? s[0] : (lane == 1 ? s[1] : s[2]);
    if (A.Omega && lane >= 3 && lane < 6) A.Omega[3 * (size_t)dst + lane - 3] = lane == 3 ? s[3] : (lane == 4 ? s[4] : s[5]);
    __syncwarp();
  }
}

GridGeom make_geom(const dp_plan* P) {
  GridGeom g;
  g.nx = P->p.nx; g.ny = P->p.ny; g.nz = P->p.nz; g.w = P->p.w; g.wall_mode = P->p.wall_mode;
  g.nbx = P->nbx; g.nby = P->nby;
  g.Lx = P->p.Lx; g.Ly = P->p.Ly; g.H = P->p.H; g.h = P->h; g.alpha = P->alpha;
  return g;
}

size_t spread_smem_bytes(int nz) {
  return sizeof(double) * ((size_t)3 * nz * TY * TX + nz + 2 * PCH * DP_MAX_W + (size_t)PCH * nz + PCH * 3) + sizeof(int) * PCH * 4;
}

}  // namespace

cudaError_t dp_launch_bin(dp_plan* P, int n, const double* pos, const double* force, const double* torque, cudaStream_t st) {
  GridGeom g = make_geom(P);
  cudaError_t e = cudaMemsetAsync(P->d_bin_count, 0, sizeof(int) * P->nbins, st);
  if (e != cudaSuccess) return e;
  e = cudaMemsetAsync(P->d_flag, 0, sizeof(int), st);
  if (e != cudaSuccess) return e;
  const int T = 256, B = (n + T - 1) / T;
  k_bin_count<<<B, T, 0, st>>>(n, pos, g, P->d_bin_of, P->d_slot_of, P->d_bin_count, P->d_flag);
  k_scan<<<1, 1024, 0, st>>>(P->nbins, P->d_bin_count, P->d_bin_start);
  k_bin_scatter<<<B, T, 0, st>>>(n, pos, force, torque, g, P->d_bin_of, P->d_slot_of, P->d_bin_start, P->d_perm, P->d_pos_s,
                                P->d_frc_s, P->fields == 6 ? P->d_trq_s : nullptr);
  return cudaGetLastError();
}

cudaError_t dp_launch_spread(dp_plan* P, int n, bool with_force, bool with_torque, cudaStream_t st) {
  (void)n; (void)with_force;
  SpreadArgs A;
  A.g = make_geom(P);
  A.pos_s = P->d_pos_s;
  A.val_s[0] = P->d_frc_s; A.val_s[1] = P->d_trq_s;
  A.beta[0] = P->p.beta_M; A.beta[1] = P->p.beta_D;
  A.Z[0] = P->ZM; A.Z[1] = P->ZD;
  A.field0[0] = 0; A.field0[1] = 3;
  A.ngroups = with_torque ? 2 : 1;
  A.bin_start = P->d_bin_start;
  A.znodes = P->d_znodes;
  A.grid = P->d_real;
  A.real_field = P->real_field;
  size_t smem = spread_smem_bytes(P->p.nz);
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(k_spread, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  dim3 grid(P->nbins, A.ngroups);
  k_spread<<<grid, SPREAD_THREADS, smem, st>>>(A);
  return cudaGetLastError();
}

cudaError_t dp_launch_interp(dp_plan* P, int n, double* U, double* Omega, cudaStream_t st) {
  InterpArgs A;
  A.g = make_geom(P);
  A.pos_s = P->d_pos_s; A.perm = P->d_perm;
  A.beta[0] = P->p.beta_M; A.beta[1] = P->p.beta_D;
  A.Z[0] = P->ZM; A.Z[1] = P->ZD;
  A.znodes = P->d_znodes; A.zweights = P->d_zweights;
  A.grid = P->d_real; A.real_field = P->real_field;
  A.U = U; A.Omega = Omega;
  int blocks = (n + INTERP_WARPS - 1) / INTERP_WARPS;
  const int maxb = 148 * 64;
  if (blocks > maxb) blocks = maxb;
  if (blocks < 1) blocks = 1;
  k_interp<<<blocks, INTERP_WARPS * 32, 0, st>>>(n, A);
  return cudaGetLastError();
}
