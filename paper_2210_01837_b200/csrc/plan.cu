// plan.cu — C ABI of the DP Stokes library: plan creation (tables, buffers, FFT tables or cuFFT plans), the apply pipeline
// (paper steps 1-8), host-buffer entry point, profiling and test hooks.  See include/dp.h.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "common.cuh"

namespace {

typedef long double ld;
const ld PI_LD = 3.141592653589793238462643383279502884L;

// Z = int_{-alpha}^{alpha} exp(beta (sqrt(1 - (s/alpha)^2) - 1)) ds  (eq 54).
// s = alpha sin(theta) makes the integrand alpha exp(beta (cos(theta) - 1)) cos(theta), analytic on [-pi/2, pi/2]:
// composite 16-point Gauss-Legendre on 32 panels (Newton on the three-term recurrence for the nodes).
double es_norm_host(double alpha, double beta) {
  const int NP = 16, PANELS = 32;
  ld x[NP], w[NP];
  for (int i = 0; i < NP; ++i) {
    ld t = cosl(PI_LD * (i + 0.75L) / (NP + 0.5L)), dp = 1;
    for (int it = 0; it < 60; ++it) {
      ld p0 = 1, p1 = t;
      for (int k = 2; k <= NP; ++k) { ld p2 = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
      dp = NP * (t * p1 - p0) / (t * t - 1);
      ld dt = p1 / dp; t -= dt;
      if (fabsl(dt) < 1e-20L) break;
    }
    ld p0 = 1, p1 = t;
    for (int k = 2; k <= NP; ++k) { ld p2 = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
    dp = NP * (t * p1 - p0) / (t * t - 1);
    x[i] = t; w[i] = 2 / ((1 - t * t) * dp * dp);
  }
  ld sum = 0;
  const ld a = -PI_LD / 2, width = PI_LD / PANELS;
  for (int p = 0; p < PANELS; ++p)
    for (int i = 0; i < NP; ++i) {
      ld th = a + width * (p + 0.5L * (x[i] + 1));
      sum += 0.5L * width * w[i] * expl((ld)beta * (cosl(th) - 1)) * cosl(th);
    }
  return (double)((ld)alpha * sum);
}

// Gauss-Legendre nodes / weights on [-1, 1] by Newton on the three-term recurrence
void gl_rule(int n, std::vector<ld>& x, std::vector<ld>& w) {
  x.resize(n); w.resize(n);
  for (int i = 0; i < n; ++i) {
    ld t = cosl(PI_LD * (i + 0.75L) / (n + 0.5L)), dp = 1;
    for (int it = 0; it < 80; ++it) {
      ld p0 = 1, p1 = t;
      for (int k = 2; k <= n; ++k) { ld p2 = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
      dp = n * (t * p1 - p0) / (t * t - 1);
      const ld dt = p1 / dp; t -= dt;
      if (fabsl(dt) < 1e-19L) break;
    }
    ld p0 = 1, p1 = t;
    for (int k = 2; k <= n; ++k) { ld p2 = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
    dp = n * (t * p1 - p0) / (t * t - 1);
    x[i] = t; w[i] = 2 / ((1 - t * t) * dp * dp);
  }
}

// Effective hydrodynamic radius of a blob whose envelope is the tensor product phi(x) phi(y) phi(z) of the ES kernel
// (eq 53-54) in an UNBOUNDED fluid, in units of the grid spacing h (alpha = w/2).  c(beta) = R_h/h is
// intrinsic to the kernel (eq 56 and PAPER.md:362-364); the paper tabulates it in Tables I-II.
//   monopole (translation-translation self mobility 1/(6 pi eta R_h), eq 1 in Fourier space, isotropic by cubic symmetry):
//       1/(6 pi R_h) = (2/3) int_0^inf g(t)^3 dt,   g(t) = (1/pi) int_0^inf |phi^(q)|^2 exp(-q^2 t) dq,
//       phi^(q) = int phi(s) cos(q s) ds;
//   dipole (rotation-rotation self mobility 1/(8 pi eta R_h^3)):  R_h = (3/(4 pi))^{1/3} / int phi(s)^2 ds.
// Both reduce to the Gaussian relations of eq 8.
double es_radius_over_h(int w, double beta, bool dipole) {
  const ld alpha = 0.5L * w;
  const double Z = es_norm_host((double)alpha, beta);
  // nodes s = alpha sin(theta): integrands analytic in theta
  std::vector<ld> gx, gw;
  gl_rule(24, gx, gw);
  const int PANELS = 8;
  std::vector<ld> s_nodes, s_wphi;          // s_k and w_k phi(s_k) ds
  for (int p = 0; p < PANELS; ++p)
    for (size_t i = 0; i < gx.size(); ++i) {
      const ld width = PI_LD / PANELS, th = -PI_LD / 2 + width * (p + 0.5L * (gx[i] + 1));
      const ld phi = expl((ld)beta * (cosl(th) - 1)) / (ld)Z;
      s_nodes.push_back(alpha * sinl(th));
      s_wphi.push_back(0.5L * width * gw[i] * phi * alpha * cosl(th));
    }
  if (dipole) {
    ld i2 = 0;
    for (size_t k = 0; k < s_nodes.size(); ++k) {
      const ld c = sqrtl(1 - (s_nodes[k] / alpha) * (s_nodes[k] / alpha));
      i2 += s_wphi[k] * expl((ld)beta * (c - 1)) / (ld)Z;          // phi^2 ds = (phi ds) phi
    }
    return (double)(cbrtl(3 / (4 * PI_LD)) / i2);
  }
  // int_0^inf g^3 dt = int_0^1 g(t)^3 dt + int_1^inf g(t)^3 dt.  In the second part t = 1/y^2 and q = r y give
  //   g(t) = (y/pi) G(y),  G(y) = int_0^inf |phi^(r y)|^2 exp(-r^2) dr,   int_1^inf g^3 dt = (2/pi^3) int_0^1 G(y)^3 dy,
  // so both parts are integrals of smooth functions over [0, 1] (the t^{-3/2} tail is integrated exactly by the map).
  auto phihat2 = [&](ld qq) {
    ld ph = 0;
    for (size_t k = 0; k < s_nodes.size(); ++k) ph += s_wphi[k] * cosl(qq * s_nodes[k]);
    return ph * ph;
  };
  // part 1: |phi^(q)|^2 on a composite rule in q over [0, QMAX]; beyond QMAX |phi^|^2 <= (2 phi(alpha)/q)^2 ~ e^{-2 beta}
  const ld QMAX = 48.0L;
  const int QPAN = 96;
  std::vector<ld> q, p2w;                   // q_j and weight_j |phi^(q_j)|^2
  for (int p = 0; p < QPAN; ++p)
    for (size_t i = 0; i < gx.size(); ++i) {
      const ld width = QMAX / QPAN, qq = width * (p + 0.5L * (gx[i] + 1));
      q.push_back(qq); p2w.push_back(0.5L * width * gw[i] * phihat2(qq));
    }
  ld part1 = 0, part2 = 0;
  const int TPAN = 4;
  for (int p = 0; p < TPAN; ++p)
    for (size_t i = 0; i < gx.size(); ++i) {
      const ld width = 1.0L / TPAN, t = width * (p + 0.5L * (gx[i] + 1));
      ld g = 0;
      for (size_t j = 0; j < q.size(); ++j) g += p2w[j] * expl(-q[j] * q[j] * t);
      g /= PI_LD;
      part1 += 0.5L * width * gw[i] * g * g * g;
    }
  // part 2: G(y) with r in [0, RMAX] (exp(-RMAX^2) ~ 1e-22)
  const ld RMAX = 7.0L;
  const int RPAN = 7;
  for (int p = 0; p < TPAN; ++p)
    for (size_t i = 0; i < gx.size(); ++i) {
      const ld width = 1.0L / TPAN, y = width * (p + 0.5L * (gx[i] + 1));
      ld G = 0;
      for (int pr = 0; pr < RPAN; ++pr)
        for (size_t k = 0; k < gx.size(); ++k) {
          const ld wr = RMAX / RPAN, r = wr * (pr + 0.5L * (gx[k] + 1));
          G += 0.5L * wr * gw[k] * phihat2(r * y) * expl(-r * r);
        }
      part2 += 0.5L * width * gw[i] * G * G * G;
    }
  const ld integ = part1 + 2 * part2 / (PI_LD * PI_LD * PI_LD);
  return (double)(1 / (6 * PI_LD * (2.0L / 3.0L) * integ));
}

// Truncation point of the ES kernel's derivative (footnote 47): |phi'(s)| ~ e^{beta c} sqrt(1 - c^2)/c with
// c = sqrt(1 - (s/alpha)^2) is stationary where c (1 - c^2) = 1/beta; of the two roots in (0, 1) the smaller one is the minimum
// of |phi'| next to the edge of the support, beyond which the derivative blows up.  Newton from c = 1/beta; returns
// u = |s|/alpha = sqrt(1 - c^2), or a negative number when beta <= 3 sqrt(3)/2 (no interior minimum).
double es_dphi_cut_host(double beta) {
  if (!(beta > 2.598076211353316)) return -1.0;
  const ld rhs = 1 / (ld)beta;
  ld c = rhs;
  for (int it = 0; it < 100; ++it) {
    const ld f = c - c * c * c - rhs, df = 1 - 3 * c * c;
    const ld dc = f / df;
    c -= dc;
    if (fabsl(dc) < 1e-21L) break;
  }
  return (double)sqrtl((1 - c) * (1 + c));
}

void set_err(dp_plan* P, const char* what, const char* detail) {
  if (P) P->last_error = std::string(what) + ": " + (detail ? detail : "");
}

#define CK(call)                                                           \
  do {                                                                     \
    cudaError_t e__ = (call);                                              \
    if (e__ != cudaSuccess) { set_err(P, #call, cudaGetErrorString(e__)); return DP_ECUDA; } \
  } while (0)
#define CKF(call)                                                          \
  do {                                                                     \
    cufftResult r__ = (call);                                              \
    if (r__ != CUFFT_SUCCESS) { char b__[64]; snprintf(b__, sizeof b__, "cufft error %d", (int)r__); set_err(P, #call, b__); return DP_ECUFFT; } \
  } while (0)

// makes the plan's device current for the lifetime of the guard and restores the caller's device afterwards
struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; cudaGetLastError(); }
    if (prev != dev) ok = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

template <class T> int dev_alloc(dp_plan* P, T** ptr, size_t count) {
  cudaError_t e = cudaMalloc((void**)ptr, sizeof(T) * (count ? count : 1));
  if (e != cudaSuccess) { set_err(P, "cudaMalloc", cudaGetErrorString(e)); cudaGetLastError(); return DP_ENOMEM; }
  P->device_bytes += sizeof(T) * (count ? count : 1);
  return DP_OK;
}

int make_fft(dp_plan* P) {
  const int nx = P->p.nx, ny = P->p.ny;
  long long n[2] = {ny, nx};
  long long rembed[2] = {ny, nx}, cembed[2] = {ny, P->nkxp};
  const long long batch = 3LL * P->p.nz;           // one field triple per call
  size_t ws_f = 0, ws_i = 0;
  CKF(cufftCreate(&P->fft_fwd));
  CKF(cufftCreate(&P->fft_inv));
  P->fft_ok = true;
  CKF(cufftSetAutoAllocation(P->fft_fwd, 0));
  CKF(cufftSetAutoAllocation(P->fft_inv, 0));
  CKF(cufftMakePlanMany64(P->fft_fwd, 2, n, rembed, 1, (long long)ny * nx, cembed, 1, (long long)ny * P->nkxp, CUFFT_D2Z, batch, &ws_f));
  CKF(cufftMakePlanMany64(P->fft_inv, 2, n, cembed, 1, (long long)ny * P->nkxp, rembed, 1, (long long)ny * nx, CUFFT_Z2D, batch, &ws_i));
  P->fft_work_bytes = ws_f > ws_i ? ws_f : ws_i;
  if (P->fft_work_bytes) {
    cudaError_t e = cudaMalloc(&P->d_fft_work, P->fft_work_bytes);
    if (e != cudaSuccess) { set_err(P, "cudaMalloc(cufft work)", cudaGetErrorString(e)); cudaGetLastError(); return DP_ENOMEM; }
    P->device_bytes += P->fft_work_bytes;
  }
  CKF(cufftSetWorkArea(P->fft_fwd, P->d_fft_work));
  CKF(cufftSetWorkArea(P->fft_inv, P->d_fft_work));
  return DP_OK;
}

int run_pipeline(dp_plan* P, int n, const double* pos, const double* force, const double* torque, double* U, double* Omega,
                 cudaStream_t st, int last_stage) {
  const bool with_torque = torque != nullptr;
  // kernel-derivative torque mode: torques ride in the force field and Omega is gathered from u: three fields throughout
  const bool torque_field = with_torque && !P->kernel_torque;
  const bool want_omega = !P->kernel_torque && (Omega != nullptr || (last_stage < 5 && P->fields == 6 && last_stage >= 3));
  const bool prof = P->profiling && P->ev_ok;
  P->last_stream = st;
  P->ev_recorded = false;
  if (prof) CK(cudaEventRecord(P->ev[0], st));
  // the zero planes are skipped only with the own FFT passes (cuFFT transforms every plane) and only in full products
  // (the test hooks hand out whole grids)
  const bool dense = P->p.dense_planes || !P->own_fft || last_stage < 5;
  CK(dp_launch_bin(P, n, pos, force, torque, dense, st));
  if (prof) CK(cudaEventRecord(P->ev[1], st));
  CK(dp_launch_spread(P, n, true, with_torque, st));
  if (prof) CK(cudaEventRecord(P->ev[2], st));
  if (last_stage >= 2) {
    if (P->own_fft) {
      CK(dp_fft_own_forward(P, torque_field ? 6 : 3, st));
    } else {
      CKF(cufftSetStream(P->fft_fwd, st));
      CKF(cufftExecD2Z(P->fft_fwd, P->d_real, (cufftDoubleComplex*)P->d_cplx));
      if (torque_field) CKF(cufftExecD2Z(P->fft_fwd, P->d_real + 3 * P->real_field, (cufftDoubleComplex*)(P->d_cplx + 3 * P->cplx_field)));
    }
  }
  if (prof) CK(cudaEventRecord(P->ev[3], st));
  if (last_stage >= 3) CK(dp_launch_solve(P, torque_field, want_omega, st));
  if (prof) CK(cudaEventRecord(P->ev[4], st));
  if (last_stage >= 4) {
    if (P->own_fft) {
      CK(dp_fft_own_inverse(P, want_omega ? 6 : 3, st));
    } else {
      CKF(cufftSetStream(P->fft_inv, st));
      CKF(cufftExecZ2D(P->fft_inv, (cufftDoubleComplex*)P->d_cplx, P->d_real));
      if (want_omega) CKF(cufftExecZ2D(P->fft_inv, (cufftDoubleComplex*)(P->d_cplx + 3 * P->cplx_field), P->d_real + 3 * P->real_field));
    }
  }
  if (prof) CK(cudaEventRecord(P->ev[5], st));
  if (last_stage >= 5) CK(dp_launch_interp(P, n, U, Omega, st));
  if (prof) { CK(cudaEventRecord(P->ev[6], st)); P->ev_recorded = true; }
  return DP_OK;
}

int check_apply_args(dp_plan* P, int n, const double* pos, const double* force, const double* torque, const double* U, const double* Omega) {
  if (!P) return DP_EINVAL;
  if (n < 0 || n > P->p.max_particles) { set_err(P, "dp_mobility_apply", "n out of range"); return DP_EINVAL; }
  if (n == 0) return DP_OK;                      // nothing to do; pointers of empty arrays may legitimately be NULL
  if (n > 0 && (!pos || !U)) { set_err(P, "dp_mobility_apply", "pos and U are required"); return DP_EINVAL; }
  if (!force && !torque) { set_err(P, "dp_mobility_apply", "force and torque both NULL"); return DP_EINVAL; }
  if ((torque || Omega) && !P->torques) { set_err(P, "dp_mobility_apply", "plan created with use_torques = 0"); return DP_EINVAL; }
  return DP_OK;
}

}  // namespace

// device staging buffers of dp_mobility_apply_host: owned by the plan (dp_plan::host_stage), allocated on first use, all or nothing
struct dp_host_stage {
  double *pos = nullptr, *frc = nullptr, *trq = nullptr, *U = nullptr, *Om = nullptr;
  cudaStream_t st = nullptr;
  size_t bytes = 0;
  void release() {
    void* hb[] = {pos, frc, trq, U, Om};
    for (void* b : hb) if (b) cudaFree(b);
    if (st) cudaStreamDestroy(st);
    pos = frc = trq = U = Om = nullptr; st = nullptr; bytes = 0;
  }
};

extern "C" {

double dp_es_norm(double alpha, double beta) { return es_norm_host(alpha, beta); }

double dp_es_radius_over_h(int w, double beta, int dipole) {
  if (w < 1 || !(beta > 0) || (dipole != 0 && dipole != 1)) return -1.0;
  return es_radius_over_h(w, beta, dipole != 0);
}

int dp_supported_nz(int* out, int cap) { return dp_solve_nz_list(out, cap); }

double dp_es_dphi_cut(double beta) { return es_dphi_cut_host(beta); }

const char* dp_strerror(int code) {
  switch (code) {
    case DP_OK: return "ok";
    case DP_EINVAL: return "invalid argument";
    case DP_ENOMEM: return "out of device memory";
    case DP_ECUDA: return "CUDA error";
    case DP_ECUFFT: return "cuFFT error";
    case DP_EDOMAIN: return "particle outside the domain";
    case DP_ETOOBIG: return "problem larger than the fixed work array (dp_bin_particles_static: use a plan)";
    default: return "unknown error";
  }
}

const char* dp_last_error(const dp_plan* P) { return P ? P->last_error.c_str() : "null plan"; }
size_t dp_device_bytes(const dp_plan* P) { return P ? P->device_bytes : 0; }
int dp_complex_row_pitch(const dp_plan* P) { return P ? P->nkxp : 0; }

int dp_destroy(dp_plan* P) {
  if (!P) return DP_OK;
  DeviceGuard guard(P->p.device);
  cudaDeviceSynchronize();
  if (P->fft_ok) { cufftDestroy(P->fft_fwd); cufftDestroy(P->fft_inv); }
  dp_fft_own_destroy(P);
  void* bufs[] = {P->d_real, P->d_cplx, P->d_fft_work, P->d_znodes, P->d_zweights, P->d_pos_s, P->d_frc_s, P->d_trq_s, P->d_perm, P->d_meta, P->d_wrec,
                  P->d_bin_of, P->d_slot_of, P->d_bin_count, P->d_bin_start, P->d_scan_sums, P->d_tile_cnt, P->d_tile_list, P->d_ov_tiles, P->d_ov_count, P->d_flag, P->d_lmin};
  for (void* b : bufs) if (b) cudaFree(b);
  if (P->ev_ok) { for (auto& e : P->ev) cudaEventDestroy(e); for (auto& e : P->ev_fft) cudaEventDestroy(e); }
  if (P->host_stage) {
    dp_host_stage* hs = static_cast<dp_host_stage*>(P->host_stage);
    hs->release();
    delete hs;
  }
  dp_solve_destroy_tables(P);
  delete P;
  return DP_OK;
}

int dp_create(const dp_params* prm, dp_plan** out) {
  if (!out) return DP_EINVAL;
  *out = nullptr;
  if (!prm) return DP_EINVAL;
  const dp_params& p = *prm;
  if (p.wall_mode != DP_BOTTOM_WALL && p.wall_mode != DP_SLIT) return DP_EINVAL;
  if (!(p.Lx > 0) || !(p.Ly > 0) || !(p.H > 0) || !(p.eta > 0)) return DP_EINVAL;
  if (p.w < 4 || p.w > DP_MAX_W) return DP_EINVAL;
  if (p.nx < DP_TILE_X + p.w || p.ny < DP_TILE_Y + p.w || (p.nx & 1) || (p.ny & 1)) return DP_EINVAL;
  if (!dp_solve_supports_nz(p.nz)) return DP_EINVAL;
  const double hx = p.Lx / p.nx, hy = p.Ly / p.ny;
  if (fabs(hx - hy) > 1e-12 * hx) return DP_EINVAL;
  if (!(p.beta_M > 0) || (p.use_torques && !(p.beta_D > 0))) return DP_EINVAL;
  if (p.max_particles < 1) return DP_EINVAL;
  if (p.fft_backend != 0 && p.fft_backend != 1) return DP_EINVAL;
  if (p.transfer_fp32 != 0 && p.transfer_fp32 != 1) return DP_EINVAL;
  if (p.dense_planes != 0 && p.dense_planes != 1) return DP_EINVAL;
  if (p.torque_mode != 0 && p.torque_mode != 1) return DP_EINVAL;
  if (p.solve_kernel != 0 && p.solve_kernel != 1) return DP_EINVAL;
  if (!(p.slip_0 >= 0) || !(p.slip_H >= 0) || !std::isfinite(p.slip_0) || !std::isfinite(p.slip_H)) return DP_EINVAL;
  for (int c = 0; c < 2; ++c) if (!std::isfinite(p.uwall_0[c]) || !std::isfinite(p.uwall_H[c])) return DP_EINVAL;
  if (p.wall_mode == DP_BOTTOM_WALL && (p.slip_0 != 0 || p.slip_H != 0 || p.uwall_H[0] != 0 || p.uwall_H[1] != 0)) return DP_EINVAL;
  if (p.use_torques && p.torque_mode == 1 && es_dphi_cut_host(p.beta_D) < 0) return DP_EINVAL;   // phi' has no minimum to truncate at
  if (p.transfer_fp32 && !(p.fft_backend == 0 && dp_fft_own_supported(p.nx, p.ny))) return DP_EINVAL;   // fp32 grids are read by the own x passes only
  if (p.wall_mode == DP_SLIT && p.w * hx > p.H) return DP_EINVAL;     // a kernel may overlap one wall, not both
  if ((double)p.nz * p.ny * (p.nx + 16) >= 2.0e9) return DP_EINVAL;    // 32-bit plane indexing inside the kernels

  dp_plan* P = new (std::nothrow) dp_plan();
  if (!P) return DP_ENOMEM;
  P->p = p;
  P->h = hx;
  P->alpha = 0.5 * p.w * hx;
  P->ZM = es_norm_host(P->alpha, p.beta_M);
  P->ZD = p.use_torques ? es_norm_host(P->alpha, p.beta_D) : 1.0;
  P->nkx = p.nx / 2 + 1;
  P->nkxp = (P->nkx + 7) / 8 * 8;
  P->torques = p.use_torques != 0;
  P->kernel_torque = P->torques && p.torque_mode == 1;
  P->solve_force_tile = p.solve_kernel == 1;
  P->fields = (P->torques && !P->kernel_torque) ? 6 : 3;
  P->nrec = P->torques ? (P->kernel_torque ? 3 : 2) : 1;
  P->ucutD = P->kernel_torque ? es_dphi_cut_host(p.beta_D) : 1.0;
  P->nbx = (p.nx + DP_TILE_X - 1) / DP_TILE_X;
  P->nby = (p.ny + DP_TILE_Y - 1) / DP_TILE_Y;
  P->nbins = P->nbx * P->nby;
  P->real_field = (size_t)p.nz * p.ny * p.nx;
  P->own_fft = p.fft_backend == 0 && dp_fft_own_supported(p.nx, p.ny);
  P->cplx_field = P->own_fft ? dp_fft_own_cplx_field(P) : (size_t)p.nz * p.ny * P->nkxp;

  int rc = DP_OK;
  DeviceGuard guard(p.device);
  if (!guard.ok) { cudaGetLastError(); delete P; return DP_ECUDA; }
  cudaError_t ce = cudaSuccess;
#define TRY(x) do { rc = (x); if (rc != DP_OK) { std::string msg = P->last_error; dp_destroy(P); (void)msg; return rc; } } while (0)
  TRY(dev_alloc(P, &P->d_real, p.transfer_fp32 ? (P->real_field * P->fields + 1) / 2 : P->real_field * P->fields));   // fp32 grids: half the bytes
  TRY(dev_alloc(P, &P->d_cplx, P->cplx_field * P->fields));
  TRY(dev_alloc(P, &P->d_znodes, (size_t)p.nz));
  TRY(dev_alloc(P, &P->d_zweights, (size_t)p.nz));
  const size_t np = (size_t)p.max_particles;
  TRY(dev_alloc(P, &P->d_pos_s, 3 * np));
  TRY(dev_alloc(P, &P->d_frc_s, 3 * np));
  if (p.use_torques) TRY(dev_alloc(P, &P->d_trq_s, 3 * np));
  TRY(dev_alloc(P, &P->d_perm, np));
  TRY(dev_alloc(P, &P->d_meta, np));
  TRY(dev_alloc(P, &P->d_wrec, np * P->nrec * (2 * DP_MAX_W + p.nz)));
  TRY(dev_alloc(P, &P->d_bin_of, np));
  TRY(dev_alloc(P, &P->d_slot_of, np));
  TRY(dev_alloc(P, &P->d_bin_count, (size_t)P->nbins));
  TRY(dev_alloc(P, &P->d_bin_start, (size_t)P->nbins + 1));
  TRY(dev_alloc(P, &P->d_scan_sums, (size_t)P->nbins / 8192 + 1));
  TRY(dev_alloc(P, &P->d_tile_cnt, (size_t)P->nbins));
  TRY(dev_alloc(P, &P->d_tile_list, (size_t)P->nbins * 40));
  TRY(dev_alloc(P, &P->d_ov_tiles, (size_t)P->nbins));
  TRY(dev_alloc(P, &P->d_ov_count, (size_t)1));
  TRY(dev_alloc(P, &P->d_flag, (size_t)1));
  TRY(dev_alloc(P, &P->d_lmin, (size_t)1));
  {   // device shape, once per plan: grid sizes of the persistent kernels and the shared-memory limit their attributes are raised to
    int sms = 0, optin = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, p.device) != cudaSuccess ||
        cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, p.device) != cudaSuccess || sms < 1) {
      set_err(P, "cudaDeviceGetAttribute", "cannot query the device"); cudaGetLastError(); dp_destroy(P); return DP_ECUDA;
    }
    P->sm_count = sms; P->smem_optin = optin;
    cudaError_t te = dp_transfer_setup(P);
    if (te != cudaSuccess) { set_err(P, "dp_transfer_setup", cudaGetErrorString(te)); cudaGetLastError(); dp_destroy(P); return DP_ECUDA; }
  }
  if (P->own_fft) {
    cudaError_t fe = dp_fft_own_create(P);
    if (fe != cudaSuccess) { set_err(P, "dp_fft_own_create", cudaGetErrorString(fe)); dp_destroy(P); return DP_ECUDA; }
  } else {
    TRY(make_fft(P));
  }

  // tables: nodes z_l and quadrature weights h^2 (H/2) w_l, w_l Clenshaw-Curtis:
  //   w_l = (2/N)(1/c~_l) sum_{n even} (1/c~_n) (2/(1-n^2)) cos(n l pi/N)
  {
    const int nz = p.nz, N = nz - 1;
    std::vector<double> zn(nz), zw(nz);
    for (int l = 0; l < nz; ++l) {
      zn[l] = 0.5 * p.H * (1.0 + cos(M_PI * l / N));
      ld sum = 0;
      for (int n = 0; n <= N; n += 2) {
        ld cn = (n == 0 || n == N) ? 2 : 1;
        sum += (2 / (1 - (ld)n * n)) / cn * cosl(PI_LD * n * l / N);
      }
      ld cl = (l == 0 || l == N) ? 2 : 1;
      zw[l] = (double)((ld)(hx * hx * 0.5 * p.H) * (2 / (ld)N) / cl * sum);
    }
    cudaError_t e1 = cudaMemcpy(P->d_znodes, zn.data(), sizeof(double) * nz, cudaMemcpyHostToDevice);
    cudaError_t e2 = cudaMemcpy(P->d_zweights, zw.data(), sizeof(double) * nz, cudaMemcpyHostToDevice);
    cudaError_t e3 = dp_solve_upload_tables(P);
    if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess) { dp_destroy(P); return DP_ECUDA; }
  }
  {
    bool ok = true;
    for (auto& e : P->ev) ok = ok && (cudaEventCreate(&e) == cudaSuccess);
    for (auto& e : P->ev_fft) ok = ok && (cudaEventCreate(&e) == cudaSuccess);
    P->ev_ok = ok;
  }
  ce = cudaDeviceSynchronize();
  if (ce != cudaSuccess) { dp_destroy(P); return DP_ECUDA; }
#undef TRY
  *out = P;
  return DP_OK;
}

int dp_mobility_apply(dp_plan* P, int n, const double* pos, const double* force, const double* torque, double* U, double* Omega,
                      void* cuda_stream) {
  int rc = check_apply_args(P, n, pos, force, torque, U, Omega);
  if (rc != DP_OK) return rc;
  if (n == 0) return DP_OK;
  DeviceGuard guard(P->p.device);
  if (!guard.ok) { set_err(P, "cudaSetDevice", "cannot select the plan's device"); cudaGetLastError(); return DP_ECUDA; }
  return run_pipeline(P, n, pos, force, torque, U, Omega, (cudaStream_t)cuda_stream, 5);
}

int dp_debug_run_stage(dp_plan* P, int n, const double* pos, const double* force, const double* torque, int last_stage, void* cuda_stream) {
  double dummy = 0;
  int rc = check_apply_args(P, n, pos, force, torque, &dummy, nullptr);
  if (rc != DP_OK) return rc;
  if (last_stage < 1 || last_stage > 4 || n == 0) return DP_EINVAL;
  DeviceGuard guard(P->p.device);
  if (!guard.ok) { cudaGetLastError(); return DP_ECUDA; }
  return run_pipeline(P, n, pos, force, torque, nullptr, nullptr, (cudaStream_t)cuda_stream, last_stage);
}

int dp_check(dp_plan* P) {
  if (!P) return DP_EINVAL;
  DeviceGuard guard(P->p.device);
  CK(cudaStreamSynchronize(P->last_stream));
  int flag = 0;
  CK(cudaMemcpy(&flag, P->d_flag, sizeof(int), cudaMemcpyDeviceToHost));
  return flag ? DP_EDOMAIN : DP_OK;
}

int dp_set_profiling(dp_plan* P, int on) {
  if (!P) return DP_EINVAL;
  P->profiling = on != 0;
  return DP_OK;
}

int dp_stage_ms(dp_plan* P, float* ms) {
  if (!P || !ms) return DP_EINVAL;
  for (int i = 0; i < 8; ++i) ms[i] = 0.f;
  if (!P->ev_recorded) { set_err(P, "dp_stage_ms", "no profiled apply recorded"); return DP_EINVAL; }
  DeviceGuard guard(P->p.device);
  CK(cudaEventSynchronize(P->ev[6]));
  for (int i = 0; i < 6; ++i) CK(cudaEventElapsedTime(&ms[i], P->ev[i], P->ev[i + 1]));
  ms[6] = 0.f;   // the k = 0 kernel is launched inside the solve stage
  CK(cudaEventElapsedTime(&ms[7], P->ev[0], P->ev[6]));
  return DP_OK;
}

int dp_fft_pass_ms(dp_plan* P, float* ms) {
  if (!P || !ms) return DP_EINVAL;
  for (int i = 0; i < 4; ++i) ms[i] = 0.f;
  if (!P->ev_recorded || !P->own_fft) { set_err(P, "dp_fft_pass_ms", "no profiled apply with the own FFT passes recorded"); return DP_EINVAL; }
  DeviceGuard guard(P->p.device);
  CK(cudaEventSynchronize(P->ev[6]));
  CK(cudaEventElapsedTime(&ms[0], P->ev[2], P->ev_fft[0]));
  CK(cudaEventElapsedTime(&ms[1], P->ev_fft[0], P->ev[3]));
  CK(cudaEventElapsedTime(&ms[2], P->ev[4], P->ev_fft[1]));
  CK(cudaEventElapsedTime(&ms[3], P->ev_fft[1], P->ev[5]));
  return DP_OK;
}

size_t dp_buffer_bytes(const dp_plan* P, int which) {
  if (!P) return 0;
  if (which == 0) return sizeof(double) * P->real_field * P->fields;
  if (which == 1) return sizeof(double2) * (size_t)P->p.nz * P->p.ny * P->nkxp * P->fields;     // natural layout, see dp.h
  return 0;
}

int dp_fft_backend(const dp_plan* P) { return P ? (P->own_fft ? 0 : 1) : -1; }
int dp_solve_kernel(const dp_plan* P) { return P ? ((P->solve_pair_tab && !P->solve_force_tile) ? 0 : 1) : -1; }

// ---- the sort of the last product (test hook: what dp_bin_particles_static is compared with)
int dp_copy_bins_to_host(dp_plan* P, int n, int* perm, int* tile_start) {
  if (!P || !tile_start || n < 0 || n > P->p.max_particles || (n > 0 && !perm)) return DP_EINVAL;
  DeviceGuard guard(P->p.device);
  CK(cudaStreamSynchronize(P->last_stream));
  if (n > 0) CK(cudaMemcpy(perm, P->d_perm, sizeof(int) * (size_t)n, cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(tile_start, P->d_bin_start, sizeof(int) * ((size_t)P->nbins + 1), cudaMemcpyDeviceToHost));
  return DP_OK;
}

int dp_zero_planes(dp_plan* P) {
  if (!P) return DP_EINVAL;
  DeviceGuard guard(P->p.device);
  CK(cudaStreamSynchronize(P->last_stream));
  int lm = 0;
  CK(cudaMemcpy(&lm, P->d_lmin, sizeof(int), cudaMemcpyDeviceToHost));
  return lm < 0 ? 0 : (lm > P->p.nz ? P->p.nz : lm);
}

int dp_copy_buffer_to_host(dp_plan* P, int which, void* host, size_t bytes) {
  if (!P || !host) return DP_EINVAL;
  if (bytes > dp_buffer_bytes(P, which) || dp_buffer_bytes(P, which) == 0) return DP_EINVAL;
  DeviceGuard guard(P->p.device);
  CK(cudaStreamSynchronize(P->last_stream));
  if (which == 1 && P->own_fft) {
    // the own FFT passes keep the half spectrum transposed with ky digit-reversed: hand out the natural layout
    double2* tmp = nullptr;
    const size_t full = dp_buffer_bytes(P, 1);
    CK(cudaMalloc(&tmp, full));
    cudaError_t e = cudaMemsetAsync(tmp, 0, full, P->last_stream);
    if (e == cudaSuccess) e = dp_fft_own_untranspose(P, tmp, P->last_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(P->last_stream);
    if (e == cudaSuccess) e = cudaMemcpy(host, tmp, bytes, cudaMemcpyDeviceToHost);
    cudaFree(tmp);
    CK(e);
    return DP_OK;
  }
  if (which == 0 && P->p.transfer_fp32) {
    // the real grids are stored in fp32: widen on the host so that the hook always hands out doubles
    const size_t cnt = bytes / sizeof(double);
    std::vector<float> tmp(cnt);
    CK(cudaMemcpy(tmp.data(), P->d_real, cnt * sizeof(float), cudaMemcpyDeviceToHost));
    double* out = static_cast<double*>(host);
    for (size_t i = 0; i < cnt; ++i) out[i] = (double)tmp[i];
    return DP_OK;
  }
  CK(cudaMemcpy(host, which == 0 ? (const void*)P->d_real : (const void*)P->d_cplx, bytes, cudaMemcpyDeviceToHost));
  return DP_OK;
}

}  // extern "C"

// ---- one plane of an internal buffer (test hook of the full-size parity tests)
extern "C" int dp_copy_plane_to_host(dp_plan* P, int which, int field, int l, void* host, size_t bytes) {
  if (!P || !host || field < 0 || field >= P->fields || l < 0 || l >= P->p.nz) return DP_EINVAL;
  DeviceGuard guard(P->p.device);
  CK(cudaStreamSynchronize(P->last_stream));
  const size_t plane_index = (size_t)field * P->p.nz + l;
  if (which == 0) {
    const size_t cnt = (size_t)P->p.ny * P->p.nx;
    if (bytes != cnt * sizeof(double)) return DP_EINVAL;
    if (P->p.transfer_fp32) {
      std::vector<float> tmp(cnt);
      CK(cudaMemcpy(tmp.data(), reinterpret_cast<const float*>(P->d_real) + plane_index * cnt, cnt * sizeof(float), cudaMemcpyDeviceToHost));
      double* out = static_cast<double*>(host);
      for (size_t i = 0; i < cnt; ++i) out[i] = (double)tmp[i];
      return DP_OK;
    }
    CK(cudaMemcpy(host, P->d_real + plane_index * cnt, bytes, cudaMemcpyDeviceToHost));
    return DP_OK;
  }
  if (which == 1) {
    const size_t cnt = (size_t)P->p.ny * P->nkxp;
    if (bytes != cnt * sizeof(double2)) return DP_EINVAL;
    if (!P->own_fft) {
      CK(cudaMemcpy(host, P->d_cplx + plane_index * cnt, bytes, cudaMemcpyDeviceToHost));
      return DP_OK;
    }
    double2* tmp = nullptr;
    CK(cudaMalloc(&tmp, bytes));
    cudaError_t e = cudaMemsetAsync(tmp, 0, bytes, P->last_stream);
    if (e == cudaSuccess) e = dp_fft_own_untranspose_plane(P, plane_index, tmp, P->last_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(P->last_stream);
    if (e == cudaSuccess) e = cudaMemcpy(host, tmp, bytes, cudaMemcpyDeviceToHost);
    cudaFree(tmp);
    CK(e);
    return DP_OK;
  }
  return DP_EINVAL;
}

extern "C" double dp_effective_radius(const dp_plan* P, int dipole) {
  if (!P || (dipole != 0 && dipole != 1)) return -1.0;
  if (dipole && !P->torques) return -1.0;
  return P->h * es_radius_over_h(P->p.w, dipole ? P->p.beta_D : P->p.beta_M, dipole != 0);
}

// ---- host-buffer entry point -----------------------------------------------------------------------------------------
extern "C" int dp_mobility_apply_host(dp_plan* P, int n, const double* pos, const double* force, const double* torque, double* U,
                                      double* Omega) {
  int rc = check_apply_args(P, n, pos, force, torque, U, Omega);
  if (rc != DP_OK) return rc;
  if (n == 0) return DP_OK;
  DeviceGuard guard(P->p.device);
  if (!guard.ok) { set_err(P, "cudaSetDevice", "cannot select the plan's device"); cudaGetLastError(); return DP_ECUDA; }
  if (!P->host_stage) {
    dp_host_stage* fresh = new (std::nothrow) dp_host_stage();
    if (!fresh) return DP_ENOMEM;
    const size_t bytes = sizeof(double) * 3 * (size_t)P->p.max_particles;
    const int nbuf = P->torques ? 5 : 3;
    double** slots[5] = {&fresh->pos, &fresh->frc, &fresh->U, &fresh->trq, &fresh->Om};
    cudaError_t e = cudaSuccess;
    for (int i = 0; i < nbuf && e == cudaSuccess; ++i) e = cudaMalloc((void**)slots[i], bytes);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&fresh->st, cudaStreamNonBlocking);
    if (e != cudaSuccess) {                       // all or nothing: nothing half-initialised survives a failed attempt
      set_err(P, "dp_mobility_apply_host staging", cudaGetErrorString(e));
      cudaGetLastError();
      fresh->release();
      delete fresh;
      return e == cudaErrorMemoryAllocation ? DP_ENOMEM : DP_ECUDA;
    }
    fresh->bytes = (size_t)nbuf * bytes;
    P->device_bytes += fresh->bytes;
    P->host_stage = fresh;
  }
  dp_host_stage* hs = static_cast<dp_host_stage*>(P->host_stage);
  const size_t nb = sizeof(double) * 3 * (size_t)n;
  CK(cudaMemcpyAsync(hs->pos, pos, nb, cudaMemcpyHostToDevice, hs->st));
  if (force) CK(cudaMemcpyAsync(hs->frc, force, nb, cudaMemcpyHostToDevice, hs->st));
  if (torque) CK(cudaMemcpyAsync(hs->trq, torque, nb, cudaMemcpyHostToDevice, hs->st));
  rc = run_pipeline(P, n, hs->pos, force ? hs->frc : nullptr, torque ? hs->trq : nullptr, hs->U, Omega ? hs->Om : nullptr, hs->st, 5);
  if (rc != DP_OK) return rc;
  CK(cudaMemcpyAsync(U, hs->U, nb, cudaMemcpyDeviceToHost, hs->st));
  if (Omega) CK(cudaMemcpyAsync(Omega, hs->Om, nb, cudaMemcpyDeviceToHost, hs->st));
  CK(cudaStreamSynchronize(hs->st));
  return DP_OK;
}
