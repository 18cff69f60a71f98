// fft.cu — the batched 2D xy FFTs of the DP Stokes solver (paper step 2 and step 7) as two
// shared-memory passes per direction instead of a library plan:
//
//   forward   pass X: every real grid row (f, l, y, :) -> real-to-complex FFT along x -> written TRANSPOSED into the half
//                     spectrum T[f][l][kx][y]  (y contiguous)
//             pass Y: every row T[f][l][kx][:] -> complex FFT along y, in place; ky stays at its digit-reversed position
//   (per-wavenumber solve on T: it is pointwise in (kx, ky), so it only needs ky as a function of the position)
//   inverse   pass Y: inverse FFT along y in place (digit-reversed in, natural out)
//             pass X: gather T[f][l][:][y] -> complex-to-real FFT along x -> real grid row
//
// Each pass reads every grid value once and writes it once (4 passes per product and field instead of the ten of the
// library's multi-kernel plans at 4320 x 4320).  A row (or a batch of short rows) lives in shared memory for its whole
// transform (fft_engine.cuh).  One persistent CTA per SM holds the small twiddle tables and independent row slots
// (x passes: two slots of 256 threads; y passes: three slots of 160 threads — 270 / 240 / 288 lines per stage of a 4320-point
// row waste fewer thread rounds at 160 than at 256; named barriers, 128 registers per thread), so that one slot's memory phases
// overlap the other slots' butterflies.  The stage with the largest stride exchanges its data directly with global memory (coalesced: consecutive
// threads take consecutive elements); the other side of the y passes is one bulk asynchronous copy per row
// (cp.async.bulk + mbarrier), prefetched in the inverse pass; the other side of the x passes is the transposed
// scatter / gather of 16-byte elements (rb consecutive y per kx).
// The real transform of length nx is a complex transform of length M = nx/2 on z[m] = x[2m] + i x[2m+1] with the usual
// split  X[k] = E[k] + W_nx^k O[k],  E = (Z[k] + conj Z[M-k])/2,  O = -i (Z[k] - conj Z[M-k])/2.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "common.cuh"
#include "fft_engine.cuh"

namespace {

using namespace dpfft;

// slots per CTA and threads per slot of the x passes and of the y passes
#define DP_FFT_XSLOTS 2
#define DP_FFT_XTPS 256
#define DP_FFT_YSLOTS 3
#define DP_FFT_YTPS 160
#define DP_FFT_XTPS_FWD 320
// the forward x pass runs best with 320 threads per slot (its loads are one contiguous row per slot: more lines in flight), the
// inverse with 256 (its gather keeps 2 x 9 values per thread in registers at 256 threads; measured 4.7 / 5.1 ms and 6.4 / 5.5 ms at cfg 5)
constexpr int XSLOTS = DP_FFT_XSLOTS, XTPS = DP_FFT_XTPS, XTHREADS = XSLOTS * XTPS;
constexpr int XFTPS = DP_FFT_XTPS_FWD, XFTHREADS = XSLOTS * XFTPS;
#define DP_FFT_YSLOTS_FWD 2
#define DP_FFT_YTPS_FWD 288
// the forward y pass (whose first stage loads its lines from global memory into registers) runs best with two slots of 288 threads:
// every stage of a 4320-point row (270 / 240 / 288 lines) is then ONE round of its slot; measured 3.9 against 4.6 ms at cfg 5, while
// the inverse (bulk-load prefetch, stores straight to global) loses with that shape (4.2 against 3.4 ms)
constexpr int YSLOTS = DP_FFT_YSLOTS, YTPS = DP_FFT_YTPS, YTHREADS = YSLOTS * YTPS;
constexpr int YFSLOTS = DP_FFT_YSLOTS_FWD, YFTPS = DP_FFT_YTPS_FWD, YFTHREADS = YFSLOTS * YFTPS;
constexpr int SLOT_ELEMS = 4320;               // complex elements a slot can hold (69 120 bytes)

struct dp_fft_own {
  Factors Fx, Fy;            // M = nx/2 and ny
  int rbx = 1, rby = 1;      // rows per slot batch in the x and y passes
  int off_x[MAX_STAGES] = {}, off_y[MAX_STAGES] = {}, ntw_x = 0, ntw_y = 0;   // per-stage twiddle tables (fft_engine.cuh)
  double2* d_tw_x = nullptr;   // stage tables of the length-M transform
  double2* d_post_x = nullptr; // exp(-2 pi i k / nx), k <= M/2
  double2* d_tw_y = nullptr;   // stage tables of the length-ny transform
  unsigned short* d_pos_x = nullptr;   // position of Z[k] after the forward x transform
  int* d_ky_of_pos = nullptr;          // FFT-order ky index held at position p of a transformed y row
  size_t smem_x = 0, smem_y = 0, smem_y_fwd = 0;
  int grid = 148;
  void (*ky_fwd)(struct FftYArgs) = nullptr;
  void (*ky_inv)(struct FftYArgs) = nullptr;
  void (*kx_fwd)(struct FftXArgs) = nullptr;
  void (*kx_inv)(struct FftXArgs) = nullptr;
};

// ---- PTX wrappers: mbarrier, bulk asynchronous copies, named barriers
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gmem_src, unsigned bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
               "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_store(void* gmem_dst, const void* smem_src, unsigned bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gmem_dst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_proxy() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
template <int TPS> __device__ __forceinline__ void slot_barrier(int slot) { asm volatile("bar.sync %0, %1;" ::"r"(slot + 1), "n"(TPS) : "memory"); }

struct FftYArgs {
  double2* data;          // rows of n complex numbers, contiguous
  long long rows;
  const double2* tw;      // stage tables, ntw entries
  int ntw, off[MAX_STAGES];
  Factors F;
  int rb;                 // rows per slot batch
  const int* lmin;        // forward pass: planes l < *lmin of every field are zero and skipped (null: none)
  int nz, nkx, fields;    // rows = fields * nz * nkx
};

struct FftXArgs {
  double* real;           // [planes][ny][nx]
  double2* cplx;          // [planes][nkx][ny]
  long long planes;       // fields * nz
  int nx, ny, M;
  const double2* tw;      // stage tables, ntw entries
  int ntw, off[MAX_STAGES];
  const double2* post;    // length M/2 + 1
  const unsigned short* pos;
  Factors F;
  int rb;                 // rows (consecutive y) per slot batch; divides ny
  const int* lmin;        // forward pass: planes l < *lmin of every field are zero and skipped (null: none)
  int nz;                 // planes = fields * nz
};

__host__ __device__ inline size_t align16(size_t b) { return (b + 15) / 16 * 16; }

// hooks of edge_lines (called between the loads of a round and its arithmetic), plain values only
struct MidNone { __device__ __forceinline__ void operator()(int, int) const {} };
// The kernels are templates on the factorisation <R0, R1, R2> of the hot sizes (no runtime dispatch, every index into the
// argument arrays static, only three butterflies in the instruction stream); <0, 0, 0> is the general version that
// reads the radices from its arguments.
// (NN = R0 R1 R2, the transform length, is a compile-time constant there too: the index arithmetic of every line — id / (n / R) — then
// compiles to a multiplication instead of an integer division)
template <int TPS, int R0, int NN, bool INV, class Mid, class TS, class TD>
__device__ __forceinline__ void run_edge(int r0, const TS* src, TD* dst, const double2* tw1, int n, int rows, int tid, const Mid& mid) {
  if constexpr (R0 > 0) edge_lines<R0, INV>(src, dst, tw1, NN, rows, (size_t)NN, (size_t)NN, tid, TPS, mid);
  else edge_dispatch<INV>(r0, src, dst, tw1, n, rows, (size_t)n, (size_t)n, tid, TPS, mid);
}
// the shared-memory stages after (forward) or before (inverse) the edge stage, with the slot's barrier between stages;
// LAST_BARRIER: also after the final one
template <int TPS, int R0, int R1, int R2, bool INV, bool LAST_BARRIER, class FA>
__device__ __forceinline__ void run_inner(const FA& A, double2* buf, const double2* tw, int n, int rows, int tid, int slot) {
  if constexpr (R0 > 0) {
    constexpr int S1 = R2, NN = R0 * R1 * R2;    // stride of stage 1; n = R0 R1 R2 as a compile-time constant
    if (!INV) {
      stage_lines<R1, false>(buf, tw + A.off[1], NN, S1, rows, NN, tid, TPS);
      slot_barrier<TPS>(slot);
      stage_lines<R2, false>(buf, tw + A.off[2], NN, 1, rows, NN, tid, TPS);
      if (LAST_BARRIER) slot_barrier<TPS>(slot);
    } else {
      stage_lines<R2, true>(buf, tw + A.off[2], NN, 1, rows, NN, tid, TPS);
      slot_barrier<TPS>(slot);
      stage_lines<R1, true>(buf, tw + A.off[1], NN, S1, rows, NN, tid, TPS);
      if (LAST_BARRIER) slot_barrier<TPS>(slot);
    }
  } else if (!INV) {
    int S = n / A.F.r[0];
    for (int j = 1; j < A.F.ns; ++j) {
      S /= A.F.r[j];
      stage_dispatch<false>(A.F.r[j], buf, tw + A.off[j], n, S, rows, n, tid, TPS);
      if (LAST_BARRIER || j + 1 < A.F.ns) slot_barrier<TPS>(slot);
    }
  } else {
    int S = 1;
    for (int j = A.F.ns - 1; j >= 1; --j) {
      stage_dispatch<true>(A.F.r[j], buf, tw + A.off[j], n, S, rows, n, tid, TPS);
      S *= A.F.r[j];
      if (LAST_BARRIER || j > 1) slot_barrier<TPS>(slot);
    }
  }
}

// ---------------------------------------------------------------------------------------------- pass Y (in place)
// Forward: the first stage reads the row from global memory (edge_lines), the other stages run in shared memory, the
// result leaves with one bulk store; a slot waits for its previous store to have read the buffer before it starts the next
// row (the CTA's other slots are busy meanwhile).
template <int R0, int R1, int R2>
__global__ void __launch_bounds__(YFTHREADS, 1) k_fft_y_fwd(FftYArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = A.F.n;
  double2* tw = reinterpret_cast<double2*>(smem_raw);
  const int slot = threadIdx.x / YFTPS, st = threadIdx.x - slot * YFTPS;
  double2* buf = tw + A.ntw + (size_t)slot * A.rb * n;
  for (int i = threadIdx.x; i < A.ntw; i += YFTHREADS) tw[i] = A.tw[i];
  __syncthreads();
  // rows of the planes l >= lm of each field: per field one contiguous range of ra rows, cut into batches of rb
  int lm = A.lmin ? __ldg(A.lmin) : 0;
  lm = lm < 0 ? 0 : (lm > A.nz ? A.nz : lm);
  const long long ra = (long long)(A.nz - lm) * A.nkx, per_field = (ra + A.rb - 1) / A.rb;
  const long long nbatch = per_field * A.fields;
  for (long long b = (long long)blockIdx.x * YFSLOTS + slot; b < nbatch; b += (long long)gridDim.x * YFSLOTS) {
    const long long f = b / per_field, j = b - f * per_field;
    const long long row0 = (f * A.nz + lm) * A.nkx + j * A.rb;
    const int nr = (int)((ra - j * A.rb) < A.rb ? (ra - j * A.rb) : A.rb);
    double2* g = A.data + row0 * n;
    // the slot's previous bulk store must have read the buffer before this row's first stage overwrites it; waiting here (and not
    // between the loads and the arithmetic of the first round) keeps the first stage's registers free of the barrier: no spills
    if (st == 0) bulk_wait_read();
    slot_barrier<YFTPS>(slot);
    const MidNone mid;
    run_edge<YFTPS, R0, R0 * R1 * R2, false>(A.F.r[0], g, buf, tw + A.off[0], n, nr, st, mid);
    slot_barrier<YFTPS>(slot);
    run_inner<YFTPS, R0, R1, R2, false, false>(A, buf, tw, n, nr, st, slot);
    fence_async_proxy();
    slot_barrier<YFTPS>(slot);
    if (st == 0) bulk_store(g, buf, (unsigned)nr * n * 16u);
  }
  if (st == 0) bulk_wait_all();
}

// Inverse: the row arrives with one bulk load, all stages but the last run in shared memory, the last stage (largest
// stride) stores its results straight to global memory; then the slot's next bulk load is issued.
template <int R0, int R1, int R2>
__global__ void __launch_bounds__(YTHREADS, 1) k_fft_y_inv(FftYArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int n = A.F.n;
  double2* tw = reinterpret_cast<double2*>(smem_raw);
  const int slot = threadIdx.x / YTPS, st = threadIdx.x - slot * YTPS;
  double2* buf = tw + A.ntw + (size_t)slot * A.rb * n;
  uint64_t* mbar = reinterpret_cast<uint64_t*>(tw + A.ntw + (size_t)YSLOTS * A.rb * n) + slot;
  for (int i = threadIdx.x; i < A.ntw; i += YTHREADS) tw[i] = A.tw[i];
  if (st == 0) mbar_init(mbar, 1);
  fence_async_proxy();
  __syncthreads();
  unsigned phase = 0;
  // rows of the planes l >= lm of each field (the planes above every footprint are never interpolated from: their inverse transform
  // is skipped, as their forward transform was): per field one contiguous range of ra rows, cut into batches of rb
  int lm = A.lmin ? __ldg(A.lmin) : 0;
  lm = lm < 0 ? 0 : (lm > A.nz ? A.nz : lm);
  const long long ra = (long long)(A.nz - lm) * A.nkx, per_field = (ra + A.rb - 1) / A.rb;
  const long long nbatch = per_field * A.fields;
  const long long stride = (long long)gridDim.x * YSLOTS;
  auto batch = [&](long long bb, long long& row0, int& nr) {
    const long long f = bb / per_field, j = bb - f * per_field;
    row0 = (f * A.nz + lm) * A.nkx + j * A.rb;
    nr = (int)((ra - j * A.rb) < A.rb ? (ra - j * A.rb) : A.rb);
  };
  long long b = (long long)blockIdx.x * YSLOTS + slot;
  if (st == 0 && b < nbatch) {
    long long row0; int nr;
    batch(b, row0, nr);
    mbar_expect_tx(mbar, (unsigned)nr * n * 16u);
    bulk_load(buf, A.data + row0 * n, (unsigned)nr * n * 16u, mbar);
  }
  for (; b < nbatch; b += stride) {
    long long row0; int nr;
    batch(b, row0, nr);
    double2* g = A.data + row0 * n;
    mbar_wait(mbar, phase);
    phase ^= 1;
    run_inner<YTPS, R0, R1, R2, true, true>(A, buf, tw, n, nr, st, slot);
    const bool more = b + stride < nbatch;
    long long nrow0 = 0; int nnr = 0;
    if (more) batch(b + stride, nrow0, nnr);
    // the refill of the buffer is issued after the last stage (issuing it between that stage's loads and its arithmetic costs the
    // stage 200 bytes of spills per thread; the other slots of the CTA cover the load's latency)
    run_edge<YTPS, R0, R0 * R1 * R2, true>(A.F.r[0], buf, g, tw + A.off[0], n, nr, st, MidNone());
    fence_async_proxy();
    slot_barrier<YTPS>(slot);
    if (st == 0 && more) { mbar_expect_tx(mbar, (unsigned)nnr * n * 16u); bulk_load(buf, A.data + nrow0 * n, (unsigned)nnr * n * 16u, mbar); }
  }
}

// ---------------------------------------------------------------------------------------------- pass X forward
template <int R0, int R1, int R2, bool F32>
__global__ void __launch_bounds__(XFTHREADS, 1) k_fft_x_fwd(FftXArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int M = A.M, npost = M / 2 + 1;
  double2* tw = reinterpret_cast<double2*>(smem_raw);
  double2* post = tw + A.ntw;
  const int slot = threadIdx.x / XFTPS, st = threadIdx.x - slot * XFTPS;
  double2* buf = post + npost + (size_t)slot * A.rb * M;
  unsigned short* pos = reinterpret_cast<unsigned short*>(post + npost + (size_t)XSLOTS * A.rb * M);
  for (int i = threadIdx.x; i < A.ntw; i += XFTHREADS) tw[i] = A.tw[i];
  for (int i = threadIdx.x; i < M; i += XFTHREADS) pos[i] = A.pos[i];
  for (int i = threadIdx.x; i < npost; i += XFTHREADS) post[i] = A.post[i];
  __syncthreads();
  const int rb = A.rb, ny = A.ny, nkx = M + 1;
  int lm = A.lmin ? __ldg(A.lmin) : 0;
  lm = lm < 0 ? 0 : (lm > A.nz ? A.nz : lm);
  const int act = A.nz - lm, bpp = ny / rb;              // planes per field that can hold force; batches per plane
  const long long nbatch = (A.planes / A.nz) * act * bpp;
  const MidNone nomid;
  for (long long b = (long long)blockIdx.x * XSLOTS + slot; b < nbatch; b += (long long)gridDim.x * XSLOTS) {
    const long long pa = b / bpp;                        // index among the active planes
    const int y0 = (int)(b - pa * bpp) * rb;
    const long long pl = (pa / act) * A.nz + lm + pa % act;
    const long long row0 = pl * ny + y0;                 // flat row index over (plane, y)
    // a real row of nx doubles is read as M complex numbers z[m] = x[2m] + i x[2m+1]
    if constexpr (F32) run_edge<XFTPS, R0, R0 * R1 * R2, false>(A.F.r[0], reinterpret_cast<const float2*>(reinterpret_cast<const float*>(A.real) + row0 * A.nx), buf, tw + A.off[0], M, rb, st, nomid);
    else run_edge<XFTPS, R0, R0 * R1 * R2, false>(A.F.r[0], reinterpret_cast<const double2*>(A.real + row0 * A.nx), buf, tw + A.off[0], M, rb, st, nomid);
    slot_barrier<XFTPS>(slot);
    run_inner<XFTPS, R0, R1, R2, false, true>(A, buf, tw, M, rb, st, slot);
    // split into the spectra of the real rows and write them transposed: T[pl][kx][y0 + r]
    double2* out = A.cplx + (size_t)pl * nkx * ny + y0;
    auto split = [&](int k, int r, int Mc) {
      const int km = (k == 0) ? 0 : Mc - k;
      const double2 z1 = buf[r * Mc + pos[k]], z2 = buf[r * Mc + pos[km]];
      const double2 E = make_double2(0.5 * (z1.x + z2.x), 0.5 * (z1.y - z2.y));
      const double2 O = make_double2(0.5 * (z1.y + z2.y), -0.5 * (z1.x - z2.x));
      const double2 B = cmul(O, post[k]);
      out[(size_t)k * ny + r] = cadd(E, B);
      if (2 * k != Mc) out[(size_t)(Mc - k) * ny + r] = make_double2(E.x - B.x, -(E.y - B.y));
    };
    if constexpr (R0 > 0) {                     // static kernels: M and the rows per batch are compile-time constants (no integer division)
      constexpr int Ms = R0 * R1 * R2, RB = SLOT_ELEMS / Ms > 0 ? SLOT_ELEMS / Ms : 1;
      for (int idx = st; idx < (Ms / 2 + 1) * RB; idx += XFTPS) split(idx / RB, idx % RB, Ms);
    } else {
      for (int idx = st; idx < npost * rb; idx += XFTPS) { const int k = idx / rb; split(k, idx - k * rb, M); }
    }
    slot_barrier<XFTPS>(slot);                                  // every read of buf is done before the next batch overwrites it
  }
}

// ---------------------------------------------------------------------------------------------- pass X inverse
template <int R0, int R1, int R2, bool F32>
__global__ void __launch_bounds__(XTHREADS, 1) k_fft_x_inv(FftXArgs A) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int M = A.M, npost = M / 2 + 1;
  double2* tw = reinterpret_cast<double2*>(smem_raw);
  double2* post = tw + A.ntw;
  const int slot = threadIdx.x / XTPS, st = threadIdx.x - slot * XTPS;
  double2* buf = post + npost + (size_t)slot * A.rb * M;
  unsigned short* pos = reinterpret_cast<unsigned short*>(post + npost + (size_t)XSLOTS * A.rb * M);
  for (int i = threadIdx.x; i < A.ntw; i += XTHREADS) tw[i] = A.tw[i];
  for (int i = threadIdx.x; i < M; i += XTHREADS) pos[i] = A.pos[i];
  for (int i = threadIdx.x; i < npost; i += XTHREADS) post[i] = A.post[i];
  __syncthreads();
  const int rb = A.rb, ny = A.ny, nkx = M + 1;
  int lm = A.lmin ? __ldg(A.lmin) : 0;                   // planes l < lm are never interpolated from: not transformed back
  lm = lm < 0 ? 0 : (lm > A.nz ? A.nz : lm);
  const int act = A.nz - lm, bpp = ny / rb;
  const long long nbatch = (A.planes / A.nz) * act * bpp;
  const MidNone nomid;
  for (long long b = (long long)blockIdx.x * XSLOTS + slot; b < nbatch; b += (long long)gridDim.x * XSLOTS) {
    const long long pa = b / bpp;                        // index among the active planes
    const int y0 = (int)(b - pa * bpp) * rb;
    const long long pl = (pa / act) * A.nz + lm + pa % act;
    const long long row0 = pl * ny + y0;
    const double2* in = A.cplx + (size_t)pl * nkx * ny + y0;
    // Z'[k] = (X[k] + conj X[M-k]) + i conj(W^k) (X[k] - conj X[M-k]) at its digit-reversed position (unnormalised C2R).
    // All of a thread's gathered values are loaded before any is used: one round of global latency per batch.
    auto put = [&](int k, int r, double2 X1, double2 X2) {
      if (k == 0) {
        buf[r * M + pos[0]] = make_double2(X1.x + X2.x, X1.x - X2.x);      // imaginary parts of X[0], X[M] are ignored
      } else {
        const double2 Aa = make_double2(X1.x + X2.x, X1.y - X2.y), D = make_double2(X1.x - X2.x, X1.y + X2.y);
        const double2 Bq = cmulc(D, post[k]);
        buf[r * M + pos[k]] = make_double2(Aa.x - Bq.y, Aa.y + Bq.x);
        if (2 * k != M) buf[r * M + pos[M - k]] = make_double2(Aa.x + Bq.y, Bq.x - Aa.y);
      }
    };
    if constexpr (R0 > 0) {
      constexpr int Ms = R0 * R1 * R2, RB = SLOT_ELEMS / Ms, ITEMS = (Ms / 2 + 1) * RB, NIT = (ITEMS + XTPS - 1) / XTPS;
      double2 X1[NIT], X2[NIT];
#pragma unroll
      for (int i = 0; i < NIT; ++i) {
        const int idx = st + i * XTPS, k = idx / RB, r = idx - k * RB;
        if (idx < ITEMS) { X1[i] = __ldg(in + (size_t)k * ny + r); X2[i] = __ldg(in + (size_t)(Ms - k) * ny + r); }
      }
#pragma unroll
      for (int i = 0; i < NIT; ++i) {
        const int idx = st + i * XTPS, k = idx / RB, r = idx - k * RB;
        if (idx < ITEMS) put(k, r, X1[i], X2[i]);
      }
    } else {
#pragma unroll 4
      for (int idx = st; idx < npost * rb; idx += XTPS) {
        const int k = idx / rb, r = idx - k * rb;
        put(k, r, __ldg(in + (size_t)k * ny + r), __ldg(in + (size_t)(M - k) * ny + r));
      }
    }
    slot_barrier<XTPS>(slot);
    run_inner<XTPS, R0, R1, R2, true, true>(A, buf, tw, M, rb, st, slot);
    // last stage: results go straight to the real grid rows (z[m] = x[2m] + i x[2m+1])
    if constexpr (F32) run_edge<XTPS, R0, R0 * R1 * R2, true>(A.F.r[0], (const double2*)buf, reinterpret_cast<float2*>(reinterpret_cast<float*>(A.real) + row0 * A.nx), tw + A.off[0], M, rb, st, nomid);
    else run_edge<XTPS, R0, R0 * R1 * R2, true>(A.F.r[0], (const double2*)buf, reinterpret_cast<double2*>(A.real + row0 * A.nx), tw + A.off[0], M, rb, st, nomid);
    slot_barrier<XTPS>(slot);                                  // the stage has read buf before the next batch refills it
  }
}

// test hook: transposed, digit-reversed half spectrum -> natural layout [planes][ny][nkxp]
__global__ void k_fft_untranspose(const double2* __restrict__ T, double2* __restrict__ out, const int* __restrict__ ky_of_pos, int ny, int nkx,
                                  int nkxp, long long planes) {
  const long long total = planes * nkx * ny;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
    const int p = (int)(i % ny);
    const long long q = i / ny;
    const int kx = (int)(q % nkx);
    const long long pl = q / nkx;
    out[(pl * ny + ky_of_pos[p]) * nkxp + kx] = T[i];
  }
}


// kernel selection: the static instantiations cover the three-stage factorisations of the benchmark sizes
// (4320: 16.18.15, 2160: 16.9.15, 1080: 8.9.15, 540: 4.9.15); anything else runs the general kernel
#define DP_FFT_STATIC_LIST(X) X(16, 18, 15) X(16, 9, 15) X(8, 9, 15) X(4, 9, 15) X(18, 16, 15) X(18, 8, 15)
inline bool is3(const Factors& F, int a, int b, int c) { return F.ns == 3 && F.r[0] == a && F.r[1] == b && F.r[2] == c; }
typedef void (*KernelY)(FftYArgs);
typedef void (*KernelX)(FftXArgs);
KernelY pick_y(const Factors& F, bool inv) {
#define X(a, b, c) if (is3(F, a, b, c)) return inv ? k_fft_y_inv<a, b, c> : k_fft_y_fwd<a, b, c>;
  DP_FFT_STATIC_LIST(X)
#undef X
  return inv ? k_fft_y_inv<0, 0, 0> : k_fft_y_fwd<0, 0, 0>;
}
KernelX pick_x(const Factors& F, bool inv, int rb, bool f32) {     // the static kernels assume rb = SLOT_ELEMS / M rows per batch
#define X(a, b, c)                                                                                             \
  if (is3(F, a, b, c) && rb == SLOT_ELEMS / (a * b * c))                                                       \
    return f32 ? (inv ? k_fft_x_inv<a, b, c, true> : k_fft_x_fwd<a, b, c, true>) : (inv ? k_fft_x_inv<a, b, c, false> : k_fft_x_fwd<a, b, c, false>);
  DP_FFT_STATIC_LIST(X)
#undef X
  return f32 ? (inv ? k_fft_x_inv<0, 0, 0, true> : k_fft_x_fwd<0, 0, 0, true>) : (inv ? k_fft_x_inv<0, 0, 0, false> : k_fft_x_fwd<0, 0, 0, false>);
}

template <class T> cudaError_t upload(T** dst, const std::vector<T>& v, dp_plan* P) {
  cudaError_t e = cudaMalloc((void**)dst, sizeof(T) * v.size());
  if (e != cudaSuccess) return e;
  P->device_bytes += sizeof(T) * v.size();
  return cudaMemcpy(*dst, v.data(), sizeof(T) * v.size(), cudaMemcpyHostToDevice);
}

size_t smem_bytes_y(int n, int ntw, int rb, int slots) { return sizeof(double2) * ((size_t)ntw + (size_t)slots * rb * n) + 8 * slots; }
size_t smem_bytes_x(int M, int ntw, int rb) {
  return sizeof(double2) * ((size_t)ntw + (M / 2 + 1) + (size_t)XSLOTS * rb * M) + align16(sizeof(unsigned short) * M) + 8 * XSLOTS;
}


}  // namespace

bool dp_fft_own_supported(int nx, int ny) {
  Factors F;
  if (nx % 2 || nx / 2 > SLOT_ELEMS / 2 || ny > SLOT_ELEMS || ny % 2) return false;
  return factorize(nx / 2, &F) && factorize(ny, &F);
}

size_t dp_fft_own_cplx_field(const dp_plan* P) { return (size_t)P->p.nz * (P->p.nx / 2 + 1) * P->p.ny; }
const int* dp_fft_own_ky_table(const dp_plan* P) { return P->fft_own ? static_cast<const dp_fft_own*>(P->fft_own)->d_ky_of_pos : nullptr; }

void dp_fft_own_destroy(dp_plan* P) {
  dp_fft_own* O = static_cast<dp_fft_own*>(P->fft_own);
  if (!O) return;
  void* bufs[] = {O->d_tw_x, O->d_post_x, O->d_tw_y, O->d_pos_x, O->d_ky_of_pos};
  for (void* b : bufs) if (b) cudaFree(b);
  delete O;
  P->fft_own = nullptr;
}

cudaError_t dp_fft_own_create(dp_plan* P) {
  typedef long double ld;
  const ld PI = 3.141592653589793238462643383279502884L;
  const int nx = P->p.nx, ny = P->p.ny, M = nx / 2;
  dp_fft_own* O = new dp_fft_own();
  P->fft_own = O;
  if (!factorize(M, &O->Fx) || !factorize(ny, &O->Fy)) return cudaErrorInvalidValue;
  // rows per slot batch: as many as fit the slot; in the x passes the batch must tile a plane's ny rows
  O->rby = SLOT_ELEMS / ny < 1 ? 1 : SLOT_ELEMS / ny;
  int rbmax = SLOT_ELEMS / M;                // <= 2 rows at nx = 4320: a batch is rb * nx doubles = rb * M complex
  if (rbmax < 1) rbmax = 1;
  if (rbmax > 64) rbmax = 64;
  O->rbx = 1;
  for (int r = rbmax; r >= 1; --r) if (ny % r == 0) { O->rbx = r; break; }
  O->ntw_x = stage_tables(O->Fx, O->off_x, nullptr, true);
  O->ntw_y = stage_tables(O->Fy, O->off_y, nullptr, true);
  std::vector<double2> twx(O->ntw_x + 1), post(M / 2 + 1), twy(O->ntw_y + 1);
  stage_tables(O->Fx, O->off_x, twx.data(), true);
  stage_tables(O->Fy, O->off_y, twy.data(), true);
  for (int k = 0; k <= M / 2; ++k) post[k] = make_double2((double)cosl(2 * PI * k / nx), (double)-sinl(2 * PI * k / nx));
  std::vector<unsigned short> posx(M);
  for (int k = 0; k < M; ++k) posx[k] = (unsigned short)position_of(O->Fx, k);
  std::vector<int> kyp(ny);
  for (int k = 0; k < ny; ++k) kyp[position_of(O->Fy, k)] = k;
  cudaError_t e;
  if ((e = upload(&O->d_tw_x, twx, P)) != cudaSuccess) return e;
  if ((e = upload(&O->d_post_x, post, P)) != cudaSuccess) return e;
  if ((e = upload(&O->d_tw_y, twy, P)) != cudaSuccess) return e;
  if ((e = upload(&O->d_pos_x, posx, P)) != cudaSuccess) return e;
  if ((e = upload(&O->d_ky_of_pos, kyp, P)) != cudaSuccess) return e;
  O->smem_x = smem_bytes_x(M, O->ntw_x, O->rbx);
  O->smem_y = smem_bytes_y(ny, O->ntw_y, O->rby, YSLOTS);
  O->smem_y_fwd = smem_bytes_y(ny, O->ntw_y, O->rby, YFSLOTS);   // its own size: what the slots do not need stays L1 cache for the first stage's loads
  if (O->smem_x > 227 * 1024 || O->smem_y > 227 * 1024) return cudaErrorInvalidValue;
  O->ky_fwd = pick_y(O->Fy, false); O->ky_inv = pick_y(O->Fy, true);
  O->kx_fwd = pick_x(O->Fx, false, O->rbx, P->p.transfer_fp32 != 0); O->kx_inv = pick_x(O->Fx, true, O->rbx, P->p.transfer_fp32 != 0);
  // The limit is a property of the FUNCTION on this device, not of the plan, and plans of different grid sizes share the general kernels
  // k_fft_*<0,0,0>: every plan raises it to the device's opt-in maximum, so a plan created later with a smaller grid cannot lower it under
  // a live plan that needs more (the size a launch actually asks for is what decides the shared-memory carve-out).
  int smem_optin = 0;
  if ((e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, P->p.device)) != cudaSuccess) return e;
  if ((size_t)smem_optin < O->smem_x || (size_t)smem_optin < O->smem_y) return cudaErrorInvalidValue;
  if ((e = cudaFuncSetAttribute(O->ky_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(O->ky_inv, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(O->kx_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
  if ((e = cudaFuncSetAttribute(O->kx_inv, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
  int sms = 0;
  if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, P->p.device)) != cudaSuccess) return e;
  O->grid = sms > 0 ? sms : 148;
  return cudaSuccess;
}

static FftXArgs x_args(dp_plan* P, int nfields) {
  dp_fft_own* O = static_cast<dp_fft_own*>(P->fft_own);
  FftXArgs A;
  A.real = P->d_real; A.cplx = P->d_cplx; A.planes = (long long)nfields * P->p.nz;
  A.nx = P->p.nx; A.ny = P->p.ny; A.M = P->p.nx / 2;
  A.tw = O->d_tw_x; A.ntw = O->ntw_x; A.post = O->d_post_x; A.pos = O->d_pos_x; A.F = O->Fx; A.rb = O->rbx;
  A.lmin = P->d_lmin; A.nz = P->p.nz;
  for (int j = 0; j < MAX_STAGES; ++j) A.off[j] = O->off_x[j];
  return A;
}
static FftYArgs y_args(dp_plan* P, int nfields) {
  dp_fft_own* O = static_cast<dp_fft_own*>(P->fft_own);
  FftYArgs A;
  A.data = P->d_cplx; A.rows = (long long)nfields * P->p.nz * (P->p.nx / 2 + 1);
  A.tw = O->d_tw_y; A.ntw = O->ntw_y; A.F = O->Fy; A.rb = O->rby;
  A.lmin = P->d_lmin; A.nz = P->p.nz; A.nkx = P->p.nx / 2 + 1; A.fields = nfields;
  for (int j = 0; j < MAX_STAGES; ++j) A.off[j] = O->off_y[j];
  return A;
}
static int grid_for(const dp_fft_own* O, long long nbatch, int nslot) {
  const long long need = (nbatch + nslot - 1) / nslot;
  return (int)(need < O->grid ? (need < 1 ? 1 : need) : O->grid);
}

cudaError_t dp_fft_own_forward(dp_plan* P, int nfields, cudaStream_t st) {
  dp_fft_own* O = static_cast<dp_fft_own*>(P->fft_own);
  const FftXArgs X = x_args(P, nfields);
  O->kx_fwd<<<grid_for(O, X.planes * (X.ny / X.rb), XSLOTS), XFTHREADS, O->smem_x, st>>>(X);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (P->profiling && P->ev_ok && (e = cudaEventRecord(P->ev_fft[0], st)) != cudaSuccess) return e;
  const FftYArgs Y = y_args(P, nfields);
  O->ky_fwd<<<grid_for(O, (Y.rows + Y.rb - 1) / Y.rb, YFSLOTS), YFTHREADS, O->smem_y_fwd, st>>>(Y);
  return cudaGetLastError();
}

cudaError_t dp_fft_own_inverse(dp_plan* P, int nfields, cudaStream_t st) {
  dp_fft_own* O = static_cast<dp_fft_own*>(P->fft_own);
  const FftYArgs Y = y_args(P, nfields);
  O->ky_inv<<<grid_for(O, (Y.rows + Y.rb - 1) / Y.rb, YSLOTS), YTHREADS, O->smem_y, st>>>(Y);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (P->profiling && P->ev_ok && (e = cudaEventRecord(P->ev_fft[1], st)) != cudaSuccess) return e;
  const FftXArgs X = x_args(P, nfields);
  O->kx_inv<<<grid_for(O, X.planes * (X.ny / X.rb), XSLOTS), XTHREADS, O->smem_x, st>>>(X);
  return cudaGetLastError();
}

cudaError_t dp_fft_own_untranspose_plane(dp_plan* P, size_t plane_index, double2* dst, cudaStream_t st) {
  dp_fft_own* O = static_cast<dp_fft_own*>(P->fft_own);
  const size_t plane = (size_t)(P->p.nx / 2 + 1) * P->p.ny;
  k_fft_untranspose<<<1024, 256, 0, st>>>(P->d_cplx + plane_index * plane, dst, O->d_ky_of_pos, P->p.ny, P->p.nx / 2 + 1, P->nkxp, 1);
  return cudaGetLastError();
}

cudaError_t dp_fft_own_untranspose(dp_plan* P, double2* dst, cudaStream_t st) {
  dp_fft_own* O = static_cast<dp_fft_own*>(P->fft_own);
  k_fft_untranspose<<<1024, 256, 0, st>>>(P->d_cplx, dst, O->d_ky_of_pos, P->p.ny, P->p.nx / 2 + 1, P->nkxp, (long long)P->fields * P->p.nz);
  return cudaGetLastError();
}
