// lanczos.cu — Brownian "velocities" g = M^{1/2} W by the Lanczos iteration in the Krylov subspace of the mobility operator
// (paper Sec. V B), on top of dp_mobility_apply:
//
//     v_1 = W/|W|;   n = 1, 2, ...:   w = M v_n - beta_{n-1} v_{n-1};  alpha_n = w.v_n;  w -= alpha_n v_n;  beta_n = |w|;
//     v_{n+1} = w/beta_n;   T_n = tridiag(beta, alpha, beta);   g_n = |W| V_n T_n^{1/2} e_1;
//     eps_n = |g_n - g_{n-1}| / |g_{n-1}|  (Fig. 11);  stop when eps_n < tol.
//
// The vectors live in HBM ([F; tau] stacked: 3n or 6n doubles; the basis V_n is kept, a few tens of vectors); every product is one
// dp_mobility_apply; the vector updates and dot products are small kernels of this file (fixed-order two-stage reductions:
// deterministic); the n x n tridiagonal eigenproblem (n <= 64) is solved on the host by cyclic Jacobi rotations in long double.
// Since V_n has orthonormal columns, |g_n - g_{n-1}| = |W| |c_n - (c_{n-1}, 0)| with c_n = T_n^{1/2} e_1: the stopping rule costs no
// pass over the big vectors.  No reorthogonalisation (the paper's use stops at 1e-3, where it is not needed).
#include <cmath>
#include <vector>

#include "common.cuh"

namespace {

constexpr int RED_BLOCKS = 296, RED_THREADS = 256;

__device__ __forceinline__ double block_sum(double v) {
  __shared__ double s[RED_THREADS / 32];
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
  if (threadIdx.x < 32) {
    t = threadIdx.x < RED_THREADS / 32 ? s[threadIdx.x] : 0.0;
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  }
  __syncthreads();
  return t;            // valid in thread 0
}

// w -= c * x (skipped when x is null); partial[b] = sum over the block's elements of w * y  (y null: y = the updated w, i.e. |w|^2)
__global__ void __launch_bounds__(RED_THREADS) k_axpy_dot(size_t m, double* __restrict__ w, const double* __restrict__ x, double c,
                                                          const double* __restrict__ y, double* __restrict__ partial) {
  double acc = 0.0;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < m; i += (size_t)gridDim.x * blockDim.x) {
    double v = w[i];
    if (x) { v = fma(-c, x[i], v); w[i] = v; }
    acc = fma(v, y ? y[i] : v, acc);
  }
  const double t = block_sum(acc);
  if (threadIdx.x == 0) partial[blockIdx.x] = t;
}

__global__ void __launch_bounds__(RED_THREADS) k_finish_sum(int nb, const double* __restrict__ partial, double* __restrict__ out) {
  double acc = 0.0;
  for (int i = threadIdx.x; i < nb; i += blockDim.x) acc += partial[i];      // fixed order per thread, fixed tree: deterministic
  const double t = block_sum(acc);
  if (threadIdx.x == 0) *out = t;
}

__global__ void k_scale_copy(size_t m, double* __restrict__ dst, const double* __restrict__ src, double c) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < m; i += (size_t)gridDim.x * blockDim.x) dst[i] = c * src[i];
}

// g = sum_j coef[j] V_j  (V: [nv][m])
__global__ void k_combine(size_t m, int nv, const double* __restrict__ V, const double* __restrict__ coef, double* __restrict__ g) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < m; i += (size_t)gridDim.x * blockDim.x) {
    double acc = 0.0;
    for (int j = 0; j < nv; ++j) acc = fma(coef[j], V[(size_t)j * m + i], acc);
    g[i] = acc;
  }
}

typedef long double ld;

// c = T^{1/2} e_1 for the symmetric tridiagonal T = tridiag(beta, alpha, beta) of order n: eigen-decomposition by cyclic Jacobi
// rotations (n <= 64, long double), c = Q sqrt(max(Lambda, 0)) Q^T e_1
void sqrt_first_column(int n, const std::vector<double>& alpha, const std::vector<double>& beta, std::vector<double>& c) {
  std::vector<ld> A((size_t)n * n, 0), Q((size_t)n * n, 0);
  for (int i = 0; i < n; ++i) {
    A[(size_t)i * n + i] = alpha[i]; Q[(size_t)i * n + i] = 1;
    if (i + 1 < n) { A[(size_t)i * n + i + 1] = beta[i]; A[(size_t)(i + 1) * n + i] = beta[i]; }
  }
  for (int sweep = 0; sweep < 60; ++sweep) {
    ld off = 0, diag = 0;
    for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) { if (i != j) off += A[(size_t)i * n + j] * A[(size_t)i * n + j]; else diag += A[(size_t)i * n + i] * A[(size_t)i * n + i]; }
    if (off <= 1e-38L * (diag > 0 ? diag : 1)) break;
    for (int p = 0; p < n - 1; ++p)
      for (int q = p + 1; q < n; ++q) {
        const ld apq = A[(size_t)p * n + q];
        if (apq == 0) continue;
        const ld theta = (A[(size_t)q * n + q] - A[(size_t)p * n + p]) / (2 * apq);
        const ld t = (theta >= 0 ? 1 : -1) / (fabsl(theta) + sqrtl(theta * theta + 1));
        const ld cs = 1 / sqrtl(t * t + 1), sn = t * cs;
        for (int k = 0; k < n; ++k) {           // A <- A J
          const ld akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q];
          A[(size_t)k * n + p] = cs * akp - sn * akq; A[(size_t)k * n + q] = sn * akp + cs * akq;
        }
        for (int k = 0; k < n; ++k) {           // A <- J^T A
          const ld apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k];
          A[(size_t)p * n + k] = cs * apk - sn * aqk; A[(size_t)q * n + k] = sn * apk + cs * aqk;
        }
        for (int k = 0; k < n; ++k) {           // Q <- Q J
          const ld qkp = Q[(size_t)k * n + p], qkq = Q[(size_t)k * n + q];
          Q[(size_t)k * n + p] = cs * qkp - sn * qkq; Q[(size_t)k * n + q] = sn * qkp + cs * qkq;
        }
      }
  }
  c.assign(n, 0.0);
  for (int i = 0; i < n; ++i) {
    ld s = 0;
    for (int k = 0; k < n; ++k) {
      const ld lam = A[(size_t)k * n + k];
      s += Q[(size_t)i * n + k] * sqrtl(lam > 0 ? lam : 0) * Q[(size_t)0 * n + k];
    }
    c[i] = (double)s;
  }
}

}  // namespace

#define LCK(call)                                                                                         \
  do {                                                                                                    \
    cudaError_t e__ = (call);                                                                             \
    if (e__ != cudaSuccess) { P->last_error = std::string(#call) + ": " + cudaGetErrorString(e__); rc = DP_ECUDA; goto done; } \
  } while (0)

extern "C" int dp_lanczos_sqrt(dp_plan* P, int n, const double* pos, const double* W_force, const double* W_torque, double* g_U,
                               double* g_Omega, double tol, int max_iter, int* iters, double* eps_hist, void* cuda_stream) {
  if (!P || n < 1 || n > P->p.max_particles || !pos || !W_force || !g_U || !(tol > 0) || max_iter < 1 || max_iter > 64) return DP_EINVAL;
  if ((W_torque != nullptr) != (g_Omega != nullptr)) return DP_EINVAL;
  if (W_torque && !P->torques) return DP_EINVAL;
  // the recurrence needs a linear, symmetric positive definite operator: with moving walls dp_mobility_apply is affine (U = M F + wall flow)
  if (P->p.uwall_0[0] != 0 || P->p.uwall_0[1] != 0 || P->p.uwall_H[0] != 0 || P->p.uwall_H[1] != 0) {
    P->last_error = "dp_lanczos_sqrt: the plan has a non-zero wall velocity, so its product is affine, not linear; use a plan with uwall_0 = uwall_H = 0";
    return DP_EINVAL;
  }
  int prev_dev = -1;
  cudaGetDevice(&prev_dev);
  if (prev_dev != P->p.device && cudaSetDevice(P->p.device) != cudaSuccess) { cudaGetLastError(); return DP_ECUDA; }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const bool tq = W_torque != nullptr;
  const size_t half = 3 * (size_t)n, m = tq ? 2 * half : half;
  int rc = DP_OK;
  double *V = nullptr, *w = nullptr, *partial = nullptr, *scal = nullptr, *dcoef = nullptr;
  std::vector<double> alpha, beta, c_prev, c;
  double h_s = 0.0, nrmW = 0.0;
  int done_iters = 0;
  const int grid = RED_BLOCKS;

  LCK(cudaMalloc(&V, sizeof(double) * m * (size_t)(max_iter + 1)));
  LCK(cudaMalloc(&w, sizeof(double) * m));
  LCK(cudaMalloc(&partial, sizeof(double) * RED_BLOCKS));
  LCK(cudaMalloc(&scal, sizeof(double)));
  LCK(cudaMalloc(&dcoef, sizeof(double) * (size_t)(max_iter + 1)));

  // w = W (stacked), |W|, v_1 = W / |W|
  LCK(cudaMemcpyAsync(w, W_force, sizeof(double) * half, cudaMemcpyDeviceToDevice, st));
  if (tq) LCK(cudaMemcpyAsync(w + half, W_torque, sizeof(double) * half, cudaMemcpyDeviceToDevice, st));
  k_axpy_dot<<<grid, RED_THREADS, 0, st>>>(m, w, nullptr, 0.0, nullptr, partial);
  k_finish_sum<<<1, RED_THREADS, 0, st>>>(grid, partial, scal);
  LCK(cudaMemcpyAsync(&h_s, scal, sizeof(double), cudaMemcpyDeviceToHost, st));
  LCK(cudaStreamSynchronize(st));
  nrmW = sqrt(h_s);
  if (!(nrmW > 0.0)) {                         // W = 0: g = 0
    LCK(cudaMemsetAsync(g_U, 0, sizeof(double) * half, st));
    if (tq) LCK(cudaMemsetAsync(g_Omega, 0, sizeof(double) * half, st));
    goto done;
  }
  k_scale_copy<<<grid, RED_THREADS, 0, st>>>(m, V, w, 1.0 / nrmW);

  for (int it = 1; it <= max_iter; ++it) {
    double* vj = V + (size_t)(it - 1) * m;
    // w = M v_n
    rc = dp_mobility_apply(P, n, pos, vj, tq ? vj + half : nullptr, w, tq ? w + half : nullptr, st);
    if (rc != DP_OK) goto done;
    // w -= beta_{n-1} v_{n-1};  alpha_n = w . v_n
    k_axpy_dot<<<grid, RED_THREADS, 0, st>>>(m, w, it > 1 ? V + (size_t)(it - 2) * m : nullptr, it > 1 ? beta[it - 2] : 0.0, vj, partial);
    k_finish_sum<<<1, RED_THREADS, 0, st>>>(grid, partial, scal);
    LCK(cudaMemcpyAsync(&h_s, scal, sizeof(double), cudaMemcpyDeviceToHost, st));
    LCK(cudaStreamSynchronize(st));
    const double a = h_s;
    // w -= alpha_n v_n;  beta_n = |w|
    k_axpy_dot<<<grid, RED_THREADS, 0, st>>>(m, w, vj, a, nullptr, partial);
    k_finish_sum<<<1, RED_THREADS, 0, st>>>(grid, partial, scal);
    LCK(cudaMemcpyAsync(&h_s, scal, sizeof(double), cudaMemcpyDeviceToHost, st));
    LCK(cudaStreamSynchronize(st));
    const double b = sqrt(h_s > 0 ? h_s : 0.0);
    alpha.push_back(a); beta.push_back(b);
    done_iters = it;
    c_prev = c;
    sqrt_first_column(it, alpha, beta, c);
    bool stop = false;
    if (it > 1) {
      double num = 0.0, den = 0.0;
      for (int j = 0; j < it; ++j) { const double d = c[j] - (j < it - 1 ? c_prev[j] : 0.0); num += d * d; }
      for (int j = 0; j < it - 1; ++j) den += c_prev[j] * c_prev[j];
      const double eps = sqrt(num / den);
      if (eps_hist) eps_hist[it - 2] = eps;
      if (eps < tol) stop = true;
    }
    if (b <= 1e-14 * fabs(a)) stop = true;      // invariant subspace: g is exact
    if (stop || it == max_iter) break;
    k_scale_copy<<<grid, RED_THREADS, 0, st>>>(m, V + (size_t)it * m, w, 1.0 / b);
  }
  {
    std::vector<double> coef(c.size());
    for (size_t j = 0; j < c.size(); ++j) coef[j] = nrmW * c[j];
    LCK(cudaMemcpyAsync(dcoef, coef.data(), sizeof(double) * coef.size(), cudaMemcpyHostToDevice, st));
    k_combine<<<grid, RED_THREADS, 0, st>>>(m, (int)coef.size(), V, dcoef, w);
    LCK(cudaMemcpyAsync(g_U, w, sizeof(double) * half, cudaMemcpyDeviceToDevice, st));
    if (tq) LCK(cudaMemcpyAsync(g_Omega, w + half, sizeof(double) * half, cudaMemcpyDeviceToDevice, st));
    LCK(cudaStreamSynchronize(st));
  }
done:
  if (iters) *iters = done_iters;
  cudaStreamSynchronize(st);
  if (V) cudaFree(V);
  if (w) cudaFree(w);
  if (partial) cudaFree(partial);
  if (scal) cudaFree(scal);
  if (dcoef) cudaFree(dcoef);
  if (prev_dev >= 0 && prev_dev != P->p.device) cudaSetDevice(prev_dev);
  return rc;
}
