// Host check of the index logic of the FFT engine (paper_2210_01837_b200/csrc/fft_engine.cuh, fft_radix.cuh): the same
// __host__ __device__ stage functions the CUDA passes run, executed sequentially on the CPU and compared with the
// definition  X[k] = sum_n x[n] exp(-2 pi i n k / N)  evaluated in long double.  Compiled and run by
// tests/test_fft_engine_host.py (nvcc, no GPU needed).  Prints one line per length: n, forward error of the plain
// stages, forward error of the edge-stage variant, round-trip error of both inverse variants.
#include <complex>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "../paper_2210_01837_b200/csrc/fft_engine.cuh"

using namespace dpfft;
typedef std::complex<long double> cld;
struct NoMid { void operator()(int, int) const {} };

int main(int argc, char** argv) {
  const long double PI = 3.141592653589793238462643383279502884L;
  for (int a = 1; a < argc; ++a) {
    const int n = atoi(argv[a]);
    Factors F;
    if (!factorize(n, &F)) { printf("%d unsupported\n", n); continue; }
    int off[MAX_STAGES], offe[MAX_STAGES];
    std::vector<double2> tw(stage_tables(F, off, nullptr) + 1), twe(stage_tables(F, offe, nullptr, true) + 1);
    stage_tables(F, off, tw.data());
    stage_tables(F, offe, twe.data(), true);
    std::vector<double2> x(n), y, ye(n), z, ze(n);
    srand(n);
    for (auto& v : x) v = make_double2(rand() / (double)RAND_MAX - 0.5, rand() / (double)RAND_MAX - 0.5);
    // forward, plain stages
    y = x;
    int S = n;
    for (int j = 0; j < F.ns; ++j) { S /= F.r[j]; stage_dispatch<false>(F.r[j], y.data(), tw.data() + off[j], n, S, 1, n, 0, 1); }
    // forward, edge stage first (out of place, recurrence twiddles)
    edge_dispatch<false>(F.r[0], x.data(), ye.data(), twe.data() + offe[0], n, 1, n, n, 0, 1, NoMid());
    S = n / F.r[0];
    for (int j = 1; j < F.ns; ++j) { S /= F.r[j]; stage_dispatch<false>(F.r[j], ye.data(), twe.data() + offe[j], n, S, 1, n, 0, 1); }
    long double e1 = 0, e2 = 0, nr = 0;
    const int step = n > 1200 ? 41 : 1;
    for (int k = 0; k < n; k += step) {
      cld s = 0;
      for (int m = 0; m < n; ++m) { const long double t = -2 * PI * (long double)((long long)k * m % n) / n; s += cld(x[m].x, x[m].y) * cld(cosl(t), sinl(t)); }
      const double2 g = y[position_of(F, k)], h = ye[position_of(F, k)];
      e1 += std::norm(s - cld(g.x, g.y)); e2 += std::norm(s - cld(h.x, h.y)); nr += std::norm(s);
    }
    // inverse of both
    z = y;
    S = 1;
    for (int j = F.ns - 1; j >= 0; --j) { stage_dispatch<true>(F.r[j], z.data(), tw.data() + off[j], n, S, 1, n, 0, 1); S *= F.r[j]; }
    S = 1;
    for (int j = F.ns - 1; j >= 1; --j) { stage_dispatch<true>(F.r[j], ye.data(), twe.data() + offe[j], n, S, 1, n, 0, 1); S *= F.r[j]; }
    edge_dispatch<true>(F.r[0], ye.data(), ze.data(), twe.data() + offe[0], n, 1, n, n, 0, 1, NoMid());
    long double r1 = 0, r2 = 0, nx = 0;
    for (int j = 0; j < n; ++j) {
      r1 += powl(z[j].x / n - x[j].x, 2) + powl(z[j].y / n - x[j].y, 2);
      r2 += powl(ze[j].x / n - x[j].x, 2) + powl(ze[j].y / n - x[j].y, 2);
      nx += x[j].x * x[j].x + x[j].y * x[j].y;
    }
    printf("%d %.3Le %.3Le %.3Le %.3Le", n, sqrtl(e1 / nr), sqrtl(e2 / nr), sqrtl(r1 / nx), sqrtl(r2 / nx));
    for (int j = 0; j < F.ns; ++j) printf(" %d", F.r[j]);
    printf("\n");
  }
  return 0;
}
