// common.cuh — plan structure and shared device helpers of the DP Stokes CUDA library (sm_100a).
// Nothing here is shared with oracle/ (the CPU oracle is written independently from the paper).
#pragma once

#include <cuda_runtime.h>
#include <cufft.h>

#include <cstddef>
#include <cstdint>
#include <string>

#include "../../include/dp.h"

#define DP_MAX_NZ 64
#define DP_MAX_W 8

// xy tile of the spread kernel (grid columns per CTA); particles are binned by the tile of their footprint origin.
#define DP_TILE_X 16
#define DP_TILE_Y 4

// modes per CTA in the solve kernel (consecutive modes of one row of the half spectrum); a lane is (mode, re/im)
#define DP_SOLVE_TM 16

struct dp_tables_host;

struct dp_plan {
  dp_params p;
  // derived
  double h, alpha, ZM, ZD;      // grid spacing, ES half support, ES normalisations (eq 54)
  int nkx, nkxp;                // nx/2+1 and its padded row pitch (complex elements)
  int fields;                   // grid fields each way: 6 with torques through the Fourier-Chebyshev curl, else 3
  bool torques = false;         // torques in / Omega out allowed (dp_params.use_torques)
  bool kernel_torque = false;   // torques through the derivative of the ES kernel (dp_params.torque_mode = 1): 3 fields
  int nrec = 1;                 // weight records per particle: Delta_M [, Delta_D [, derivatives of Delta_D]]
  double ucutD = 1.0;           // |s|/alpha beyond which phi_D' is truncated to zero (footnote 47)
  int nbx, nby, nbins;          // spread tiles / particle bins
  size_t real_field, cplx_field;  // elements per field: nz*ny*nx doubles, nz*ny*nkxp double2

  // device buffers
  double* d_real = nullptr;     // [fields][nz][ny][nx]
  double2* d_cplx = nullptr;    // [fields][nz][ny][nkxp] (cuFFT path) or [fields][nz][nkx][ny] (own FFT passes)
  void* d_fft_work = nullptr;
  size_t fft_work_bytes = 0;
  double* d_znodes = nullptr;   // z_l
  double* d_zweights = nullptr; // h^2 (H/2) w_l   (quadrature weight of node l)
  // particle workspace (sorted by bin)
  double* d_pos_s = nullptr;    // [n][3] wrapped x,y and z (z < 0 marks an out-of-domain particle)
  double* d_frc_s = nullptr;    // [n][3]
  double* d_trq_s = nullptr;    // [n][3]
  int* d_perm = nullptr;        // sorted slot -> original index
  int4* d_meta = nullptr;       // sorted footprint records: wrapped origin node (i0, j0), plane range [lmin, lmax]
  double* d_wrec = nullptr;     // sorted 1-D ES weight records [nrec][max_particles][16 + nz] (transfer.cu)
  int* d_bin_of = nullptr;      // per particle
  int* d_slot_of = nullptr;     // rank within its bin
  int* d_bin_count = nullptr;   // [nbins]
  int* d_bin_start = nullptr;   // [nbins+1]
  int* d_tile_cnt = nullptr;    // [nbins] survivors per spread tile (transfer.cu: k_tile_lists)
  int* d_tile_list = nullptr;   // [nbins][40] their indices in the sorted particle arrays (the first 40)
  int* d_ov_tiles = nullptr;    // [nbins] tiles with more survivors than a staged chunk holds
  int* d_ov_count = nullptr;    // [1]
  int* d_scan_sums = nullptr;   // [ceil(nbins / 8192)] chunk totals of the two-launch scan (transfer.cu)
  int* d_flag = nullptr;        // out-of-domain flag
  int* d_lmin = nullptr;        // lowest plane index touched by any footprint of the current apply (planes below it are zero)
  size_t device_bytes = 0;
  int sm_count = 148;           // multiprocessors of the plan's device (queried once in dp_create): grid sizes of the persistent kernels
  int smem_optin = 0;           // opt-in maximum of dynamic shared memory per CTA on the plan's device

  cufftHandle fft_fwd = 0, fft_inv = 0;
  bool fft_ok = false;
  // own shared-memory FFT passes (fft.cu): half spectrum stored transposed, [field][nz][nkx][ny], ky digit-reversed
  bool own_fft = false;
  void* fft_own = nullptr;

  void* host_stage = nullptr;   // device staging buffers of dp_mobility_apply_host (plan.cu), allocated on first use
  double* d_ct_full = nullptr;  // cos(n l pi/(nz-1)) [nz][nz] for the k = 0 kernel (solve.cu), per plan
  double* d_solve_frag = nullptr;  // DMMA fragment table of the Chebyshev transforms (solve.cu), per plan
  bool solve_force_tile = false;   // dp_params.solve_kernel = 1: keep the tile kernel of solve.cu for every product (comparison runs)
  void* solve_pair_tab = nullptr;  // host copy of the tables the warp-pair solve kernel takes as a kernel parameter (solve_pair.cu)

  cudaStream_t last_stream = nullptr;
  bool profiling = false;
  cudaEvent_t ev[9] = {};
  cudaEvent_t ev_fft[2] = {};   // between the two passes of the forward / inverse xy FFT (own passes, profiling only)
  bool ev_ok = false;
  bool ev_recorded = false;
  std::string last_error;
};

// launchers implemented in transfer.cu / solve.cu; all asynchronous on `st`
cudaError_t dp_launch_bin(dp_plan* P, int n, const double* pos, const double* force, const double* torque, bool dense, cudaStream_t st);
cudaError_t dp_launch_spread(dp_plan* P, int n, bool with_force, bool with_torque, cudaStream_t st);
cudaError_t dp_launch_interp(dp_plan* P, int n, double* U, double* Omega, cudaStream_t st);
cudaError_t dp_transfer_setup(dp_plan* P);          // per plan, from dp_create: kernel attributes of the plan's spread / interpolation kernels
cudaError_t dp_launch_solve(dp_plan* P, bool with_torque_field, bool want_omega, cudaStream_t st);
cudaError_t dp_solve_upload_tables(dp_plan* P);      // per plan: constant tables, k = 0 cosine table, kernel attributes on the plan's device
void dp_solve_destroy_tables(dp_plan* P);
bool dp_solve_supports_nz(int nz);
// solve_pair.cu: the solve kernel of products with three grid fields each way (forces only / kernel-derivative torques)
bool dp_solve_pair_supports_nz(int nz);
cudaError_t dp_solve_pair_create(dp_plan* P);
void dp_solve_pair_destroy(dp_plan* P);
int dp_solve_nz_list(int* out, int cap);
// fft.cu: the xy FFTs as two shared-memory passes per direction
bool dp_fft_own_supported(int nx, int ny);
cudaError_t dp_fft_own_create(dp_plan* P);
void dp_fft_own_destroy(dp_plan* P);
size_t dp_fft_own_cplx_field(const dp_plan* P);
const int* dp_fft_own_ky_table(const dp_plan* P);
cudaError_t dp_fft_own_forward(dp_plan* P, int nfields, cudaStream_t st);
cudaError_t dp_fft_own_inverse(dp_plan* P, int nfields, cudaStream_t st);
cudaError_t dp_fft_own_untranspose(dp_plan* P, double2* dst, cudaStream_t st);
cudaError_t dp_fft_own_untranspose_plane(dp_plan* P, size_t plane_index, double2* dst, cudaStream_t st);

// ---- exponential-of-semicircle kernel, eq 54: phi(s) = exp(beta (sqrt(1-(s/alpha)^2) - 1)) / Z on |s| <= alpha
__device__ __forceinline__ double dp_es_phi(double s, double inv_alpha, double beta, double inv_Z) {
  double q = s * inv_alpha;
  double r = 1.0 - q * q;
  if (!(fabs(q) <= 1.0)) return 0.0;
  r = r < 0.0 ? 0.0 : r;
  return exp(beta * (sqrt(r) - 1.0)) * inv_Z;
}
