// fft_engine.cuh — in-place mixed-radix complex FFT of a batch of rows held in (shared) memory, fp64.
//
// N = r_1 r_2 ... r_s.  Forward = decimation in frequency (Gentleman-Sande): natural order in, digit-reversed order out;
// inverse = decimation in time (the same flow graph backwards, conjugate twiddles): digit-reversed in, natural out.
// Stage j (S = r_{j+1} ... r_s, L = r_j S): for every block b and offset m < S, the r_j elements buf[b L + t S + m]
// are one "line": a register DFT (fft_radix.cuh) and the twiddles W_L^{k m} = W_N^{(N/L) k m}, in place.  X[k] ends at
//   pos(k) = sum_j k_j N / (r_1 ... r_j),   k = k_1 + r_1 k_2 + r_1 r_2 k_3 + ...                     (digit reversal)
// Whoever consumes the spectrum pointwise (the per-wavenumber solve) reads k from the position; nothing is reordered.
// A line is one thread's work item; consecutive threads take consecutive m, so shared-memory accesses of a warp are
// contiguous 16-byte elements except in the stage with S = 1, whose stride is r_s elements (conflict free for odd r_s).
// The twiddles of an inner stage j come from that stage's own table  tw_j[(t-1) S + m] = W_L^{t m}  (t = 1..r_j-1, m < S),
// again contiguous in m.  The stage with the largest stride (j = 1) moves its data straight between global and shared
// memory (edge_lines) and generates its twiddles by recurrence from W_N^m, so all tables together are a few KB.
#pragma once

#include <cmath>

#include "fft_radix.cuh"

namespace dpfft {

constexpr int MAX_STAGES = 6;

struct Factors {
  int n;                    // transform length
  int ns;                   // number of stages
  int r[MAX_STAGES];        // radices, r[0] = r_1 is applied first in the forward transform
};

// one stage over `rows` rows of length n stored `row_stride` elements apart; tw = this stage's table (unused if S = 1)
template <int R, bool INV>
DP_HD void stage_lines(double2* __restrict__ buf, const double2* __restrict__ tw, int n, int S, int rows, int row_stride, int tid, int nth) {
  const int per_row = n / R;                 // lines per row
  const int L = R * S;
  for (int id = tid; id < rows * per_row; id += nth) {
    const int row = id / per_row, q = id - row * per_row;
    const int b = q / S, m = q - b * S;
    double2* p = buf + (size_t)row * row_stride + b * L + m;
    const double2* w = tw + m - S;           // w[t S] = W_L^{t m}
    double2 x[R];
#pragma unroll
    for (int t = 0; t < R; ++t) x[t] = p[t * S];
    if (INV) {
      if (S > 1) {
#pragma unroll
        for (int t = 1; t < R; ++t) x[t] = cmulc(x[t], w[t * S]);
      }
      Dft<R, true>::run(x);
    } else {
      Dft<R, false>::run(x);
      if (S > 1) {
#pragma unroll
        for (int t = 1; t < R; ++t) x[t] = cmul(x[t], w[t * S]);
      }
    }
#pragma unroll
    for (int t = 0; t < R; ++t) p[t * S] = x[t];
  }
}


template <bool INV>
DP_HD void stage_dispatch(int R, double2* buf, const double2* tw, int n, int S, int rows, int row_stride, int tid, int nth) {
  switch (R) {
    case 2: stage_lines<2, INV>(buf, tw, n, S, rows, row_stride, tid, nth); break;
    case 3: stage_lines<3, INV>(buf, tw, n, S, rows, row_stride, tid, nth); break;
    case 4: stage_lines<4, INV>(buf, tw, n, S, rows, row_stride, tid, nth); break;
    case 5: stage_lines<5, INV>(buf, tw, n, S, rows, row_stride, tid, nth); break;
    case 8: stage_lines<8, INV>(buf, tw, n, S, rows, row_stride, tid, nth); break;
    case 9: stage_lines<9, INV>(buf, tw, n, S, rows, row_stride, tid, nth); break;
    case 15: stage_lines<15, INV>(buf, tw, n, S, rows, row_stride, tid, nth); break;
    case 16: stage_lines<16, INV>(buf, tw, n, S, rows, row_stride, tid, nth); break;
    case 18: stage_lines<18, INV>(buf, tw, n, S, rows, row_stride, tid, nth); break;
    default: break;
  }
}

// ---- the stage with the largest stride (S = n / r_1: first forward stage, last inverse stage) straight from / to
// global memory: forward  x[t] = src[t S + m] (global, coalesced in m) -> DFT -> twiddle -> dst[t S + m] (shared);
// inverse  x[t] = src[t S + m] (shared) -> conj twiddle -> inverse DFT -> dst[t S + m] (global, coalesced).
// Its twiddles W_n^{t m} come from a recurrence on W_n^m (table tw1[m], m < S): no shared-memory traffic beyond one
// load per line.  mid(round, nrounds) is called by every thread of the group between the loads of a round and its
// arithmetic: the place where the caller synchronises buffer reuse (all rounds have the same trip count).
// src / dst may hold float2 elements (the optional fp32 real grid of the x passes): converted on load / store.
DP_HD double2 ld2(const double2* p) { return *p; }
DP_HD double2 ld2(const float2* p) { const float2 v = *p; return make_double2((double)v.x, (double)v.y); }
DP_HD void st2(double2* p, double2 v) { *p = v; }
DP_HD void st2(float2* p, double2 v) { *p = make_float2((float)v.x, (float)v.y); }

template <int R, bool INV, class Mid, class TS, class TD>
DP_HD void edge_lines(const TS* __restrict__ src, TD* __restrict__ dst, const double2* __restrict__ tw1, int n, int rows,
                      size_t src_row_stride, size_t dst_row_stride, int tid, int nth, Mid mid) {
  const int S = n / R;
  const int total = rows * S;
  const int nrounds = (total + nth - 1) / nth;
  for (int rd = 0; rd < nrounds; ++rd) {
    const int id = rd * nth + tid;
    const bool active = id < total;
    const int row = active ? id / S : 0, m = active ? id - row * S : 0;
    const TS* ps = src + row * src_row_stride + m;
    TD* pd = dst + row * dst_row_stride + m;
    double2 x[R];
    if (active) {
#pragma unroll
      for (int t = 0; t < R; ++t) x[t] = ld2(ps + t * S);
    }
    mid(rd, nrounds);
    if (active) {
      const double2 w = tw1[m];
      double2 cur = w;
      if (INV) {
#pragma unroll
        for (int t = 1; t < R; ++t) { x[t] = cmulc(x[t], cur); if (t + 1 < R) cur = cmul(cur, w); }
        Dft<R, true>::run(x);
      } else {
        Dft<R, false>::run(x);
#pragma unroll
        for (int t = 1; t < R; ++t) { x[t] = cmul(x[t], cur); if (t + 1 < R) cur = cmul(cur, w); }
      }
#pragma unroll
      for (int t = 0; t < R; ++t) st2(pd + t * S, x[t]);
    }
  }
}

template <bool INV, class Mid, class TS, class TD>
DP_HD void edge_dispatch(int R, const TS* src, TD* dst, const double2* tw1, int n, int rows, size_t src_row_stride,
                         size_t dst_row_stride, int tid, int nth, Mid mid) {
  switch (R) {
    case 2: edge_lines<2, INV>(src, dst, tw1, n, rows, src_row_stride, dst_row_stride, tid, nth, mid); break;
    case 3: edge_lines<3, INV>(src, dst, tw1, n, rows, src_row_stride, dst_row_stride, tid, nth, mid); break;
    case 4: edge_lines<4, INV>(src, dst, tw1, n, rows, src_row_stride, dst_row_stride, tid, nth, mid); break;
    case 5: edge_lines<5, INV>(src, dst, tw1, n, rows, src_row_stride, dst_row_stride, tid, nth, mid); break;
    case 8: edge_lines<8, INV>(src, dst, tw1, n, rows, src_row_stride, dst_row_stride, tid, nth, mid); break;
    case 9: edge_lines<9, INV>(src, dst, tw1, n, rows, src_row_stride, dst_row_stride, tid, nth, mid); break;
    case 15: edge_lines<15, INV>(src, dst, tw1, n, rows, src_row_stride, dst_row_stride, tid, nth, mid); break;
    case 16: edge_lines<16, INV>(src, dst, tw1, n, rows, src_row_stride, dst_row_stride, tid, nth, mid); break;
    case 18: edge_lines<18, INV>(src, dst, tw1, n, rows, src_row_stride, dst_row_stride, tid, nth, mid); break;
    default: break;
  }
}

// position of X[k] after the forward transform
DP_HD int position_of(const Factors& F, int k) {
  int p = 0, stride = F.n;
  for (int j = 0; j < F.ns; ++j) {
    stride /= F.r[j];
    p += (k % F.r[j]) * stride;
    k /= F.r[j];
  }
  return p;
}

// per-stage twiddle tables, concatenated: off[j] = start of stage j's table, returns the total number of entries.
// out (may be null to only size) receives exp(-2 pi i t m / L) at off[j] + (t-1) S + m.
// With edge = true stage 0 (handled by edge_lines) only gets its base table W_n^m, m < S.
inline int stage_tables(const Factors& F, int* off, double2* out, bool edge = false) {
  const long double PI = 3.141592653589793238462643383279502884L;
  int total = 0, S = F.n;
  for (int j = 0; j < F.ns; ++j) {
    const int R = F.r[j];
    S /= R;
    off[j] = total;
    if (S == 1 && !(edge && j == 0)) continue;
    const int L = R * S;
    if (edge && j == 0) {
      if (out)
        for (int m = 0; m < S; ++m) {
          const long double a = 2 * PI * (long double)m / L;
          out[total + m] = make_double2((double)cosl(a), (double)-sinl(a));
        }
      total += S;
      continue;
    }
    if (out)
      for (int t = 1; t < R; ++t)
        for (int m = 0; m < S; ++m) {
          const long double a = 2 * PI * (long double)((long long)t * m % L) / L;
          out[total + (t - 1) * S + m] = make_double2((double)cosl(a), (double)-sinl(a));
        }
    total += (R - 1) * S;
  }
  return total;
}

inline bool radix_supported(int r) { return r == 2 || r == 3 || r == 4 || r == 5 || r == 8 || r == 9 || r == 15 || r == 16 || r == 18; }

// Factorisation used by the passes: a large power-of-two radix first, an odd radix last (conflict-free unit-stride
// stage), as few stages as possible.  Returns false if n has a prime factor other than 2, 3, 5 or needs > MAX_STAGES.
inline bool factorize(int n, Factors* F) {
  F->n = n; F->ns = 0;
  if (n < 2) return false;
  int e2 = 0, e3 = 0, e5 = 0, m = n;
  while (m % 2 == 0) { m /= 2; ++e2; }
  while (m % 3 == 0) { m /= 3; ++e3; }
  while (m % 5 == 0) { m /= 5; ++e5; }
  if (m != 1) return false;
  int head[MAX_STAGES * 2], nh = 0, tail[MAX_STAGES * 2], nt = 0, mid[MAX_STAGES * 2], nm = 0;
  // odd radices: pair 3 with 5 -> 15 (goes last), 3 with 3 -> 9
  while (e3 > 0 && e5 > 0) { tail[nt++] = 15; --e3; --e5; }
  while (e3 >= 2) { mid[nm++] = 9; e3 -= 2; }
  // 18 = 2 * 9 absorbs one factor of two if that saves a stage (e2 = 1 mod 4 with a 9 available)
  if (nm > 0 && (e2 % 4 == 1)) { mid[nm - 1] = 18; --e2; }
  while (e3 > 0) { mid[nm++] = 3; --e3; }
  while (e5 > 0) { mid[nm++] = 5; --e5; }
  while (e2 >= 4) { head[nh++] = 16; e2 -= 4; }
  if (e2 == 3) head[nh++] = 8; else if (e2 == 2) head[nh++] = 4; else if (e2 == 1) head[nh++] = 2;
  // order: powers of two, then the other odd radices, then the 15s; make sure the last radix is odd when one exists
  for (int i = 0; i < nh; ++i) { if (F->ns >= MAX_STAGES) return false; F->r[F->ns++] = head[i]; }
  int last_odd = -1;
  for (int i = 0; i < nm; ++i) { if (F->ns >= MAX_STAGES) return false; F->r[F->ns++] = mid[i]; }
  for (int i = 0; i < nt; ++i) { if (F->ns >= MAX_STAGES) return false; F->r[F->ns++] = tail[i]; }
  for (int i = F->ns - 1; i >= 0; --i) if (F->r[i] & 1) { last_odd = i; break; }
  if (last_odd >= 0 && last_odd != F->ns - 1) { const int t = F->r[last_odd]; F->r[last_odd] = F->r[F->ns - 1]; F->r[F->ns - 1] = t; }
  int prod = 1;
  for (int i = 0; i < F->ns; ++i) prod *= F->r[i];
  return prod == n;
}

}  // namespace dpfft
