/* dp.h — C ABI of the B200-native doubly-periodic Stokes mobility product
 *
 *     (U, Omega) = M (F, tau)
 *
 * for N regularised blobs above one no-slip wall ("bottom wall") or between two ("slit channel"), doubly periodic
 * in x, y: the method of Hashemi et al., arXiv 2210.01837.  One call of dp_mobility_apply runs the paper's
 * steps 1-8 (Sec. III D) entirely in this library's hand-written CUDA kernels for sm_100a (the xy
 * FFTs included: two shared-memory passes per direction; cuFFT only when fft_backend = 1 asks for it or the grid size
 * has a prime factor > 5):
 *   step 1  spread F (and tau) with the exponential-of-semicircle kernel and wall images   eqs 7, 9, 53, 54
 *   step 2  2D FFT in xy, Chebyshev transform in z, Chebyshev differentiation
 *   step 3  per (kx,ky): pressure BVP eq 15 + BCs 17; velocity BVPs eq 18 + BCs 22, 24
 *   step 4  per (kx,ky): wall correction, eqs 42-44 (one wall) or App. A (A5),(A6),(A8),(A10) (slit)
 *   step 5  k = 0 mode, eqs 47, 51, 52 / (A12)
 *   step 6  sum, (1/2) curl u in Fourier-Chebyshev space for Omega (eq 11)
 *   step 7  inverse transforms
 *   step 8  interpolate u (and (1/2) curl u) back to the particles, eqs 10, 11
 * The exact discrete problem (grid, transforms, tau/integration BVP form, Nyquist rule, scalings) is stated in
 * DESIGN.md §2; tests compare every output with the CPU oracle in oracle/ (relative L2 <= 1e-10 in fp64).
 *
 * Conventions
 *  - All functions return DP_OK (0) or a negative error code; nothing throws across this boundary.
 *  - Particle arrays are fp64, xyz-interleaved [n][3].  "DEVICE" pointers are CUDA device pointers on the plan's
 *    device, owned by the caller, read-only for inputs, fully overwritten for outputs, never retained.
 *  - x, y may be any real number (wrapped periodically into [0,Lx) x [0,Ly)).  z must satisfy 0 <= z <= H and, for the
 *    bottom wall, z + alpha <= H with alpha = w h / 2 (kernels must not cross the open top): a
 *    particle violating this contributes nothing, receives U = Omega = 0, and is reported by dp_check().
 *  - A plan is not thread-safe: one call in flight per plan.  Plans are immutable after creation.  Every entry point
 *    that touches the device makes the plan's device current for its own duration and restores the caller's device;
 *    all device state (tables, workspaces, kernel attributes) is per plan, so plans on different devices coexist in
 *    one process.
 */
#ifndef DP_STOKES_H
#define DP_STOKES_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dp_plan dp_plan; /* opaque: owns grids, FFT tables (or cuFFT plans), solver tables, workspace */

enum { DP_BOTTOM_WALL = 0, DP_SLIT = 1 };
enum { DP_OK = 0, DP_EINVAL = -1, DP_ENOMEM = -2, DP_ECUDA = -3, DP_ECUFFT = -4, DP_EDOMAIN = -5,
       DP_ETOOBIG = -6 /* problem larger than the fixed work array of dp_bin_particles_static */ };

/* Problem statement of the paper: box doubly periodic in xy with wall(s), ES kernel (w, beta) per envelope
 * (eqs 53-54), viscosity.  The first block of fields is SURVEY.md §8(b)'s struct; the second block
 * ("extensions") was added by this build and is documented in DESIGN.md §1. */
typedef struct {
  int wall_mode;        /* DP_BOTTOM_WALL: wall at z=0, open top at z=H;  DP_SLIT: walls at z=0 and z=H   */
  double Lx, Ly, H;     /* FULL periods in x, y (reading G1); top of the Chebyshev grid                       */
  int nx, ny, nz;       /* grid: uniform in x,y (h = Lx/nx = Ly/ny to 1e-12 relative; nx, ny even), nz type-2
                           Chebyshev nodes z_l = (H/2)(1+cos(l pi/(nz-1))) including both ends;
                           only the sizes dp_supported_nz lists ({16, 19, 24, 26, 32, 40, 48, 64}: one compiled kernel set each)
                           are accepted; any other nz is DP_EINVAL                                                       */
  int w;                /* ES kernel support in cells (paper's m), 4..8; alpha = w h/2                   */
  double beta_M;        /* ES beta of the monopole envelope Delta_M (eq 54; beta, not beta/w)                            */
  double beta_D;        /* ES beta of the dipole envelope Delta_D; ignored if torques/Omega are never used               */
  double a;             /* nominal blob radius: informational only (nothing in the product depends on it, G9);
                           compare with dp_effective_radius()                                                             */
  double eta;           /* viscosity > 0                                                                                */
  int max_particles;    /* capacity of the plan's particle workspace                                                     */
  int transfer_fp32;    /* 0: everything fp64;  1: optional variant — spreading and interpolation accumulate in fp32 and
                           the real-space grids are stored in fp32 (half the bytes of steps 1, 8 and of the real side of the
                           x FFT passes); transforms and solves stay fp64.  Needs the own FFT passes (fft_backend = 0 and a
                           supported size).  Matches the fp64 product to ~1e-6 relative (tests: <= 1e-5 vs the oracle).   */
  int device;           /* CUDA device ordinal                                                                           */
  /* ---- extensions beyond SURVEY.md §8(b) ---- */
  int use_torques;      /* 0: forces in, U out only (3 grid fields); 1: also torques in / Omega out (6 fields) */
  int fft_backend;      /* 0: the library's own shared-memory FFT passes when nx, ny allow them (nx/2 and ny products
                           of 2, 3, 5; nx, ny <= 4320), else cuFFT;  1: always cuFFT (kept for comparison)                */
  int dense_planes;     /* 0 (default): planes of the Chebyshev grid above every particle's footprint hold no force, so their
                           forward transforms are identically zero; the product finds the highest touched plane while
                           binning and skips the spreading stores, forward FFT passes and solve loads of the planes above
                           it (exact: the skipped values are zeros).  1: treat every plane as dense.                        */
  int torque_mode;      /* how torques enter and Omega leaves.  0: the paper's "first way" — tau is spread as a second
                           field triple, (1/2) curl in Fourier-Chebyshev space, (1/2) curl u transformed back as a second triple
                           (6 grid fields each way);  1: its "second way" — the derivative of the ES kernel spreads
                           (1/2) curl (tau Delta_D^W) into the force field and gathers Omega = (1/2) int (u x grad Delta_D^W) from u
                           itself (3 fields each way; truncated phi', one kernel per dimension, footnotes 47-48, PAPER.md:797-798;
                           DESIGN.md reading G19).  The two discretisations agree to the method's 2-3 digits, not to roundoff;
                           mode 1 needs beta_D > 3 sqrt(3)/2.  Ignored when use_torques = 0.                                     */
  double slip_0, slip_H; /* partial slip lengths l_0, l_H >= 0 of the bottom / top wall, slit only (App. A (A1)):
                           u - u_wall = l_0 du/dz at z = 0, u - u_wall = -l_H du/dz at z = H for the tangential components; 0 = no slip.
                           The wall derivatives of the DP solution come from Chebyshev differentiation and direct summation
                           (footnote 46).  Must be 0 for DP_BOTTOM_WALL (the paper gives no slip solution there).       */
  double uwall_0[2];    /* uniform velocity (x, y) of the bottom wall (eq 27 / eq 46): enters the k = 0 column,
                           eq 52 / (A12); the product becomes affine, U = M F + (flow driven by the walls)                          */
  double uwall_H[2];    /* uniform velocity (x, y) of the top wall; slit only ((A1b), (A12)); must be 0 for DP_BOTTOM_WALL.
                           Non-uniform wall velocity fields u_wall(x, y) are not supported.                                          */
  int solve_kernel;     /* which kernel runs steps 2(z)-6 of products with three grid fields each way (forces only, or
                           torque_mode = 1).  0 (default): the register-resident warp-pair kernel (solve_pair.cu) where it is compiled
                           (nz in {16, 19, 24, 26, 32, 40, 48}), else the tile kernel;  1: always the tile kernel (solve.cu; kept for
                           comparison).  Products with six fields (torque_mode = 0 with torques) always use the tile kernel.  Both solve
                           the same discrete problem; results agree to roundoff.                                                      */
} dp_params;

/* Plan creation for the problem of PAPER.md:74 (box, walls) with the grid of PAPER.md:319 and the ES kernel of eq 54.
 * Validates, allocates (two grids of fields*nz*ny*nx doubles resp. fields*nz*(nx/2+1)*ny complex + particle workspace),
 * builds the FFT twiddle tables (or cuFFT plans), uploads the solver tables.  Synchronous.  *out = NULL on error. */
int dp_create(const dp_params* p, dp_plan** out);

/* One mobility product (U, Omega) = M (F, tau): eqs 2, 7, 10, 11 by steps 1-8 of Sec. III D
 * (PAPER.md:325-333).  Asynchronous on `cuda_stream` (a cudaStream_t; NULL = default stream).  DEVICE pointers.
 *   pos    [n][3]  positions
 *   force  [n][3]  or NULL (treated as zero)
 *   torque [n][3]  or NULL; non-NULL requires use_torques = 1
 *   U      [n][3]  required
 *   Omega  [n][3]  or NULL; non-NULL requires use_torques = 1
 * force == NULL && torque == NULL -> DP_EINVAL.  n > max_particles or n < 0 -> DP_EINVAL.  n == 0 is a no-op.
 * No host<->device copy and no synchronisation happens inside. */
int dp_mobility_apply(dp_plan* plan, int n, const double* pos, const double* force, const double* torque,
                      double* U, double* Omega, void* cuda_stream);

/* The same product (same equations) with HOST pointers: copies inputs to the device, runs dp_mobility_apply, copies U
 * (and Omega) back and synchronises.  This is the end-to-end entry point bench.py times as "e2e". */
int dp_mobility_apply_host(dp_plan* plan, int n, const double* pos, const double* force, const double* torque,
                           double* U, double* Omega);

/* Brownian "velocities" g = M^{1/2} W (Sec. V B): Lanczos iteration in the Krylov subspace of the mobility
 * operator, one dp_mobility_apply per iteration, until eps_n = |g_n - g_{n-1}| / |g_{n-1}| < tol (the quantity of Fig. 11,
 * PAPER.md:527) or max_iter (<= 64) products.  DEVICE pointers [n][3]: W_force required, W_torque or NULL (then the
 * translational block only: U = M^{tt} F); g_U required, g_Omega given iff W_torque is.  *iters receives the number of products,
 * eps_hist[0 .. *iters - 2] (HOST, may be NULL) receives eps_2, eps_3, ...  Synchronous (every iteration reads two scalars back);
 * allocates (max_iter + 2) work vectors for the duration of the call.
 * Needs n >= 1 (n == 0 is DP_EINVAL here, unlike dp_mobility_apply's no-op) and a LINEAR product: a plan with a non-zero uwall_0 / uwall_H
 * (whose product is affine, U = M F + wall-driven flow) is refused with DP_EINVAL and a dp_last_error message. */
int dp_lanczos_sqrt(dp_plan* plan, int n, const double* pos, const double* W_force, const double* W_torque, double* g_U,
                    double* g_Omega, double tol, int max_iter, int* iters, double* eps_hist, void* cuda_stream);

/* Particle binning (step a0 of the product: the counting sort by xy tile that spreading and interpolation rely on; the build's
 * own step, it is how step 1, reaches the grid without global atomics) for callers that MUST NOT ALLOCATE device
 * memory while they run.  Who that is: code living inside a host application that took all of HBM for its own memory pool when
 * it started, so that a later cudaMalloc fails or fragments the pool; a plug-in or a latency-bound loop whose host forbids driver
 * allocations after initialisation, because cudaMalloc / cudaFree may synchronise the whole device; a worker that is only ever
 * handed buffers.  dp_create gives a plan its work arrays with cudaMalloc; this entry point needs no plan and calls neither
 * cudaMalloc, cudaFree nor any library routine that allocates: the work arrays of the sort (tile and rank of every particle, tile
 * counters, scan totals; 2.5 MiB) are a fixed array inside libdpstokes.so itself, which every GPU that loads the library holds
 * until the process exits.
 *   prm         box and grid: wall_mode, Lx, Ly, H, nx, ny, w and device are used (checked as dp_create checks them), the rest ignored
 *   pos         [n][3]  DEVICE, positions (x, y wrapped periodically; a particle outside the domain in z is filed under tile 0,
 *                       as the product does before it skips it)
 *   perm        [n]     DEVICE, out: particle indices ordered by tile; the order of the particles WITHIN one tile is not fixed
 *                       (it comes from atomic counters) and may differ from call to call
 *   tile_start  [T+1]   DEVICE, out: perm[tile_start[t] .. tile_start[t+1]-1] are the particles whose w x w footprint has its
 *                       first node in tile t = ty * ceil(nx / DP_BIN_TILE_X) + tx;  T = ceil(nx/DP_BIN_TILE_X) * ceil(ny/DP_BIN_TILE_Y)
 * Limits: n <= DP_STATIC_BIN_MAX_PARTICLES and T <= DP_STATIC_BIN_MAX_TILES, else DP_ETOOBIG and nothing is launched (configs 1-4
 * fit; config 5 does not: use a plan).  Asynchronous on `cuda_stream`; inputs are read-only, outputs fully overwritten.
 * Set-up: the FIRST call on each device looks up the device address of the fixed array (cudaGetSymbolAddress, with that device
 * current) and keeps it; make that first call during your own initialisation, before any stream capture is begun.
 * Sharing: every call on a device uses the same array, which still holds the previous call's contents — the entry point clears the
 * parts that must start at zero itself (on the stream), so back-to-back calls on ONE stream are fine, but two calls that can run at
 * the same time on the GPU (different streams, different host threads) race on it and give garbage: serialise them. */
#define DP_BIN_TILE_X 16
#define DP_BIN_TILE_Y 4
#define DP_STATIC_BIN_MAX_PARTICLES 262144
#define DP_STATIC_BIN_MAX_TILES 131072
int dp_bin_particles_static(const dp_params* prm, int n, const double* pos, int* perm, int* tile_start, void* cuda_stream);

/* Test hook: the same two arrays as the LAST product of `plan` left them in the plan's own work arrays (HOST pointers; perm [n],
 * tile_start [T+1]; synchronises the last stream).  n must be the particle count of that product. */
int dp_copy_bins_to_host(dp_plan* plan, int n, int* perm, int* tile_start);

/* Domain check of the last product: "kernels must never extend outside open boundaries" (footnote 44) and
 * 0 <= z <= H.  Synchronises the last stream used; DP_EDOMAIN if any particle of the last apply was out of domain. */
int dp_check(dp_plan* plan);

/* Effective hydrodynamic radius R_h (a length, = c(beta) h) of a blob regularised by the plan's ES kernel in an unbounded
 * fluid: dipole = 0: from the translational self mobility 1/(6 pi eta R_h) of Delta_M; dipole = 1: from the rotational self
 * mobility 1/(8 pi eta R_h^3) of Delta_D (eq 8, for the Gaussian analogue; eq 56: R_h/h
 * is intrinsic to the kernel; Tables I-II, print it).  Host-side 1-D quadrature (DESIGN.md pin P1), no
 * device work.  Returns a negative number on a NULL plan or dipole = 1 on a plan without torques. */
double dp_effective_radius(const dp_plan* plan, int dipole);

/* Per-stage device times (ms) of the LAST apply, measured with CUDA events on its stream; synchronises.
 * ms[0] bin, [1] spread (step 1), [2] xy FFT forward (step 2), [3] per-wavenumber solve (z transforms + BVPs + correction +
 * curl, steps 2-6), [4] xy FFT inverse (step 7), [5] interpolate (step 8), [6] k=0 column, [7] total.
 * Only recorded if dp_set_profiling(plan, 1). */
int dp_set_profiling(dp_plan* plan, int on);
int dp_stage_ms(dp_plan* plan, float* ms /* [8] */);
/* Same, for the four kernels of the library's own xy FFT (step 2 and step 7) of the LAST profiled apply:
 * ms[0] forward x pass, [1] forward y pass, [2] inverse y pass, [3] inverse x pass.  DP_EINVAL with the cuFFT backend. */
int dp_fft_pass_ms(dp_plan* plan, float* ms /* [4] */);

/* Test hooks: copy an internal device buffer of the last apply to HOST memory (synchronises).
 *   which = 0: real grid    [fields][nz][ny][nx]       doubles  (after apply: u, (1/2) curl u in real space)
 *   which = 1: complex grid [fields][nz][ny][nkxp]     double2  (after apply: consumed by the inverse FFT, undefined;
 *              with the own FFT passes the internal layout is transposed and digit-reversed in ky — the copy undoes it)
 * dp_debug_run_stage runs the product up to and including `last_stage` (1 spread = step 1, 2 fwd FFT = step 2(xy), 3 solve =
 * steps 2(z)-6, 4 inv FFT = step 7) so that the buffers hold that stage's output.  Sizes via dp_buffer_bytes.
 * dp_copy_plane_to_host copies ONE xy plane (field, l) of buffer `which`: ny*nx doubles resp. ny*nkxp double2 in the
 * natural layout — what the full-size parity tests use to compare sampled planes and columns with the oracle. */
int dp_debug_run_stage(dp_plan* plan, int n, const double* pos, const double* force, const double* torque, int last_stage,
                       void* cuda_stream);
size_t dp_buffer_bytes(const dp_plan* plan, int which);
int dp_copy_buffer_to_host(dp_plan* plan, int which, void* host, size_t bytes);
int dp_copy_plane_to_host(dp_plan* plan, int which, int field, int l, void* host, size_t bytes);
int dp_complex_row_pitch(const dp_plan* plan); /* nkxp: padded row length (in complex numbers) of the half spectrum */
int dp_zero_planes(dp_plan* plan);             /* synchronises; number of leading planes (l = 0 is z = H) the last apply skipped */
int dp_fft_backend(const dp_plan* plan);       /* 0: own shared-memory FFT passes in use, 1: cuFFT                    */
int dp_solve_kernel(const dp_plan* plan);      /* kernel of steps 2(z)-6 for products with three grid fields each way:
                                                  0: warp-pair kernel (solve_pair.cu), 1: tile kernel (solve.cu; always used with six fields) */

/* Introspection */
double dp_es_norm(double alpha, double beta);                  /* Z of eq 54, Gauss-Legendre on the host */
double dp_es_radius_over_h(int w, double beta, int dipole);    /* c(beta) = R_h/h of eq 56 for support w and this
                                                                  beta: what dp_effective_radius divides by h; needs no plan  */
double dp_es_dphi_cut(double beta);                            /* |s|/alpha beyond which the kernel derivative of torque_mode = 1 is
                                                                  truncated to zero (footnote 47); < 0: none exists */
int dp_supported_nz(int* out, int cap);                        /* Chebyshev sizes with a compiled solve kernel; returns how many */
size_t dp_device_bytes(const dp_plan* plan);                   /* device memory owned by the plan                     */
const char* dp_strerror(int code);
const char* dp_last_error(const dp_plan* plan);                /* detail of the last failure (CUDA / cuFFT message)   */

int dp_destroy(dp_plan* plan); /* NULL is ok */

#ifdef __cplusplus
}
#endif
#endif /* DP_STOKES_H */
