// oracle/dp_oracle.cpp
//
// TEST INFRASTRUCTURE — NOT THE PRODUCT.  Plain, slow, obviously-correct CPU oracle for the
// doubly-periodic Stokes mobility product (U, Omega) = M (F, tau) of arXiv 2210.01837, written
// from the paper step by step (Sec. III D, steps 1-8) with the discrete problem pinned
// in SURVEY.md §8(c) / DESIGN.md.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call this.  It shares no code with the CUDA path (paper_2210_01837_b200/csrc).
//
// Arithmetic: fp64 everywhere; the per-wavenumber dense solves (O5, O6, O8, O9) in x87 long double with
// dense LU and partial pivoting; explicit O(n^2) DFT sums; dense Chebyshev matrices.  No blocking, no
// fusion, no fast algorithm: every function is the formula it cites, written out.
//
// Data layout: real grids [comp][l][j][i] (i = x fastest), half spectra [comp][l][ny][nkx] with
// nkx = nx/2+1, n_y in FFT order; Chebyshev index l = 0 is z = H, l = nz-1 is z = 0.
//
// Parity pins: tests/test_oracle_*.py.  Unpinned: absolute values of the
// paper's Figs. 3-8 curves (reference data not in the container) — "parity unpinned" for those only.

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;
typedef std::complex<double> cd;
typedef std::complex<long double> cld;

extern "C" {

struct or_params {
    int wall_mode;          // 0 bottom wall, 1 slit channel
    double Lx, Ly, H;       // full periods; z in [0, H]
    int nx, ny, nz;
    int w;                  // ES support in cells (paper's m), alpha = w h / 2
    double beta_M, beta_D;
    double eta;
    // App. A and eq 27/46/52: partial slip lengths of the bottom / top wall (slit only) and UNIFORM wall
    // velocities (x, y) of the bottom wall (both geometries) and of the top wall (slit); all zero = the no-slip product
    double slip_0, slip_H;
    double uwall_0[2], uwall_H[2];
};

int or_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"

static const ld PI_L = 3.141592653589793238462643383279502884L;

// ------------------------------------------------------------------------------------------------
// Gauss-Legendre nodes/weights on [-1, 1] (Newton on P_n), long double.
static void gauss_legendre(int n, std::vector<ld>& x, std::vector<ld>& w) {
    x.assign(n, 0); w.assign(n, 0);
    for (int i = 0; i < n; ++i) {
        ld t = cosl(PI_L * (i + 0.75L) / (n + 0.5L));
        ld dp = 0;
        for (int it = 0; it < 100; ++it) {
            ld p0 = 1, p1 = t;
            for (int k = 2; k <= n; ++k) { ld p2 = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
            dp = n * (t * p1 - p0) / (t * t - 1);
            ld dt = p1 / dp;
            t -= dt;
            if (fabsl(dt) < 1e-19L) break;
        }
        ld p0 = 1, p1 = t;
        for (int k = 2; k <= n; ++k) { ld p2 = ((2 * k - 1) * t * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
        dp = n * (t * p1 - p0) / (t * t - 1);
        x[i] = t; w[i] = 2 / ((1 - t * t) * dp * dp);
    }
}

extern "C" {

// Normalisation Z = int_{-alpha}^{alpha} exp(beta (sqrt(1-(s/alpha)^2) - 1)) ds   (eq 54).
// With s = alpha sin(theta): Z = alpha int_{-pi/2}^{pi/2} exp(beta (cos(theta) - 1)) cos(theta) dtheta
// (smooth integrand), 128-point Gauss-Legendre.
double or_es_norm(double alpha, double beta) {
    std::vector<ld> x, w;
    gauss_legendre(128, x, w);
    ld s = 0;
    for (size_t i = 0; i < x.size(); ++i) {
        ld th = 0.5L * PI_L * x[i];
        s += w[i] * expl((ld)beta * (cosl(th) - 1)) * cosl(th);
    }
    return (double)((ld)alpha * 0.5L * PI_L * s);
}

// phi(s; alpha, beta) of eq 54; support |s| <= alpha inclusive.
double or_es_phi(double s, double alpha, double beta, double Z) {
    double q = s / alpha;
    if (fabs(q) > 1.0) return 0.0;
    double r = 1.0 - q * q;
    if (r < 0.0) r = 0.0;
    return exp(beta * (sqrt(r) - 1.0)) / Z;
}

// Chebyshev nodes z_l = (H/2)(1 + cos(l pi/(nz-1))), l = 0..nz-1  (type-2 grid with end points)
void or_cheb_nodes(int nz, double H, double* z) {
    for (int l = 0; l < nz; ++l) z[l] = 0.5 * H * (1.0 + cos(M_PI * l / (nz - 1)));
}

// Analysis matrix A[n][l] of the DCT-I: coefficients g^_n = sum_l A[n][l] g(xi_l)  (footnote 41)
void or_cheb_analysis_matrix(int nz, double* A) {
    int N = nz - 1;
    for (int n = 0; n < nz; ++n)
        for (int l = 0; l < nz; ++l) {
            ld cn = (n == 0 || n == N) ? 2 : 1, cl = (l == 0 || l == N) ? 2 : 1;
            A[n * nz + l] = (double)((2.0L / N) / (cn * cl) * cosl(PI_L * n * l / N));
        }
}

// Synthesis matrix S[l][n] = T_n(xi_l) = cos(n l pi / (nz-1))
void or_cheb_synthesis_matrix(int nz, double* S) {
    int N = nz - 1;
    for (int l = 0; l < nz; ++l)
        for (int n = 0; n < nz; ++n) S[l * nz + n] = (double)cosl(PI_L * n * l / N);
}

}  // extern "C"

// Dense coefficient-space z-derivative: (D g^)_n = (2/H) (2/c_n) sum_{p=n+1, p-n odd} p g^_p, c_0=2, c_n=1
// (Chebyshev differentiation, step 2 PAPER.md:326; textbook formula, ref [42]).
static void cheb_diff_matrix_ld(int nz, ld H, std::vector<ld>& D) {
    D.assign((size_t)nz * nz, 0);
    for (int n = 0; n < nz; ++n)
        for (int p = n + 1; p < nz; p += 2)
            D[(size_t)n * nz + p] = (2 / H) * (n == 0 ? 1.0L : 2.0L) * p;
}

extern "C" {

void or_cheb_diff_matrix(int nz, double H, double* D) {
    std::vector<ld> Dl;
    cheb_diff_matrix_ld(nz, H, Dl);
    for (size_t i = 0; i < Dl.size(); ++i) D[i] = (double)Dl[i];
}

// Clenshaw-Curtis weights on the nodes: int_{-1}^{1} g dxi = sum_{n even} 2 g^_n/(1-n^2)
//   => w_l = sum_{n even} 2/(1-n^2) A[n][l]      (step 8 "Chebyshev quadrature")
void or_cc_weights(int nz, double* wq) {
    std::vector<double> A((size_t)nz * nz);
    or_cheb_analysis_matrix(nz, A.data());
    for (int l = 0; l < nz; ++l) {
        ld s = 0;
        for (int n = 0; n < nz; n += 2) s += 2.0L / (1.0L - (ld)n * n) * A[(size_t)n * nz + l];
        wq[l] = (double)s;
    }
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// O1 / O12: the discrete envelope S(j; i, j', l) = phi(x_i - x_j) phi(y_j' - y_j) zeta(l; z_j)
//   zeta(l; z_p) = phi(z_l - z_p) - phi(z_l + z_p) - [slit] phi(z_l - (2H - z_p))       (eqs 9, 53)
struct Footprint {
    int i0, j0;                     // first node index in x, y (unwrapped)
    std::vector<double> px, py, zeta;
};

static inline double wrap(double x, double L) { return x - floor(x / L) * L; }

static void footprint(const or_params& P, double beta, double Z, const double* z_nodes, const double* r, Footprint& fp) {
    double h = P.Lx / P.nx, alpha = 0.5 * P.w * h;
    double xw = wrap(r[0], P.Lx), yw = wrap(r[1], P.Ly);
    fp.i0 = (int)ceil((xw - alpha) / h);
    fp.j0 = (int)ceil((yw - alpha) / h);
    fp.px.resize(P.w); fp.py.resize(P.w); fp.zeta.resize(P.nz);
    for (int a = 0; a < P.w; ++a) {
        fp.px[a] = or_es_phi((fp.i0 + a) * h - xw, alpha, beta, Z);
        fp.py[a] = or_es_phi((fp.j0 + a) * h - yw, alpha, beta, Z);
    }
    double zp = r[2];
    for (int l = 0; l < P.nz; ++l) {
        double v = or_es_phi(z_nodes[l] - zp, alpha, beta, Z) - or_es_phi(z_nodes[l] + zp, alpha, beta, Z);
        if (P.wall_mode == 1) v -= or_es_phi(z_nodes[l] - (2.0 * P.H - zp), alpha, beta, Z);
        fp.zeta[l] = v;
    }
}

static inline int pmod(int i, int n) { int r = i % n; return r < 0 ? r + n : r; }

extern "C" {

// O1 spread (eq 7, step 1): grid[c][l][j][i] = sum_p val[p][c] S(p; i, j, l).  No h, no weights.
void or_spread(const or_params* P, int n, const double* pos, const double* val, double beta, double* grid) {
    size_t plane = (size_t)P->nx * P->ny, field = plane * P->nz;
    std::memset(grid, 0, sizeof(double) * 3 * field);
    double h = P->Lx / P->nx, alpha = 0.5 * P->w * h;
    double Z = or_es_norm(alpha, beta);
    std::vector<double> zn(P->nz);
    or_cheb_nodes(P->nz, P->H, zn.data());
    Footprint fp;
    for (int p = 0; p < n; ++p) {
        footprint(*P, beta, Z, zn.data(), pos + 3 * (size_t)p, fp);
        for (int c = 0; c < 3; ++c) {
            double v = val[3 * (size_t)p + c];
            for (int l = 0; l < P->nz; ++l) {
                if (fp.zeta[l] == 0.0) continue;
                for (int b = 0; b < P->w; ++b) {
                    int j = pmod(fp.j0 + b, P->ny);
                    for (int a = 0; a < P->w; ++a) {
                        int i = pmod(fp.i0 + a, P->nx);
                        grid[c * field + l * plane + (size_t)j * P->nx + i] += v * (fp.px[a] * fp.py[b] * fp.zeta[l]);
                    }
                }
            }
        }
    }
}

// O12 interpolate (eqs 10-11, step 8):
//   out[p][c] = sum_{i,j,l} grid[c][l][j][i] S(p; i, j, l) h^2 (H/2) w_l
void or_interp(const or_params* P, int n, const double* pos, const double* grid, double beta, double* out) {
    size_t plane = (size_t)P->nx * P->ny, field = plane * P->nz;
    double h = P->Lx / P->nx, alpha = 0.5 * P->w * h;
    double Z = or_es_norm(alpha, beta);
    std::vector<double> zn(P->nz), wq(P->nz);
    or_cheb_nodes(P->nz, P->H, zn.data());
    or_cc_weights(P->nz, wq.data());
#pragma omp parallel
    {
        Footprint fp;
#pragma omp for schedule(static)
        for (int p = 0; p < n; ++p) {
            footprint(*P, beta, Z, zn.data(), pos + 3 * (size_t)p, fp);
            for (int c = 0; c < 3; ++c) {
                double s = 0;
                for (int l = 0; l < P->nz; ++l) {
                    if (fp.zeta[l] == 0.0) continue;
                    double wl = h * h * (0.5 * P->H) * wq[l];
                    for (int b = 0; b < P->w; ++b) {
                        int j = pmod(fp.j0 + b, P->ny);
                        for (int a = 0; a < P->w; ++a) {
                            int i = pmod(fp.i0 + a, P->nx);
                            s += grid[c * field + l * plane + (size_t)j * P->nx + i] * (fp.px[a] * fp.py[b] * fp.zeta[l]) * wl;
                        }
                    }
                }
                out[3 * (size_t)p + c] = s;
            }
        }
    }
}

// ---- kernel-derivative torque spreading / angular-velocity interpolation (the paper's "second way", PAPER.md:335;
// footnotes 47, 48; reading G19 in DESIGN.md).  With Delta_D^W the dipole envelope of eqs 9, 53:
//   f(x_g) += (1/2) curl_x (tau Delta_D^W(x_g - r)) = (1/2) G(x_g) x tau,      G = grad_x Delta_D^W   (eq 7)
//   Omega   = (1/2) sum_g (u(x_g) x G(x_g)) h^2 (H/2) w_l                       (eq 11 integrated by parts: the adjoint)
//   G = ( phi'(x) phi(y) zeta(l),  phi(x) phi'(y) zeta(l),  phi(x) phi(y) zeta'(l) ): a different 1-D kernel along each
//   dimension (footnote 48), zeta'(l; z_p) = d/dz zeta = phi'(z_l - z_p) - phi'(z_l + z_p) - [slit] phi'(z_l - (2H - z_p)),
//   i.e. the exact z-derivative of eq 9, which makes G vanish with the particle's height ("all components of the mobility
//   go to zero at a wall", footnote 48; written with the odd kernel phi' evaluated at the mirrored distance this is the
//   positive image sign of that footnote).
// phi'(s) = -(beta s / alpha^2) phi(s) / sqrt(1 - (s/alpha)^2) is unbounded at |s| -> alpha; footnote 47: it is truncated to zero
// for |s| beyond the point where |phi'| has its minimum before it blows up.

// The cut u* = |s|/alpha of footnote 47: the stationary point of log|phi'| = beta sqrt(1-u^2) + log u - (1/2) log(1-u^2) nearest the
// edge, i.e. the root of  F(u) = -beta u/sqrt(1-u^2) + 1/u + u/(1-u^2)  in (sqrt(2/3), 1), by bisection in long double.
// Exists for beta > 3 sqrt(3)/2; returns NaN otherwise.
double or_es_dphi_cut(double beta) {
    if (!(beta > 2.5980762113533160L)) return NAN;
    auto F = [&](ld u) { ld q = 1 - u * u; return -(ld)beta * u / sqrtl(q) + 1 / u + u / q; };
    ld lo = sqrtl(2.0L / 3.0L), hi = 1 - 1e-18L;
    for (int it = 0; it < 200; ++it) {
        ld mid = 0.5L * (lo + hi);
        if (F(mid) < 0) lo = mid; else hi = mid;
    }
    return (double)(0.5L * (lo + hi));
}

// truncated derivative of eq 54's kernel (footnote 47); ucut from or_es_dphi_cut
double or_es_dphi(double s, double alpha, double beta, double Z, double ucut) {
    double q = s / alpha;
    if (fabs(q) > ucut) return 0.0;
    double r = 1.0 - q * q;
    return -(beta * s / (alpha * alpha)) * exp(beta * (sqrt(r) - 1.0)) / (sqrt(r) * Z);
}

}  // extern "C"

struct GradFootprint {
    Footprint fp;                          // phi(x), phi(y), zeta(l) of the dipole envelope
    std::vector<double> dpx, dpy, dzeta;   // phi'(x), phi'(y), zeta'(l)
};

static void grad_footprint(const or_params& P, double beta, double Z, double ucut, const double* z_nodes, const double* r, GradFootprint& g) {
    footprint(P, beta, Z, z_nodes, r, g.fp);
    double h = P.Lx / P.nx, alpha = 0.5 * P.w * h;
    double xw = wrap(r[0], P.Lx), yw = wrap(r[1], P.Ly);
    g.dpx.resize(P.w); g.dpy.resize(P.w); g.dzeta.resize(P.nz);
    for (int a = 0; a < P.w; ++a) {
        g.dpx[a] = or_es_dphi((g.fp.i0 + a) * h - xw, alpha, beta, Z, ucut);
        g.dpy[a] = or_es_dphi((g.fp.j0 + a) * h - yw, alpha, beta, Z, ucut);
    }
    double zp = r[2];
    for (int l = 0; l < P.nz; ++l) {
        double v = or_es_dphi(z_nodes[l] - zp, alpha, beta, Z, ucut) - or_es_dphi(z_nodes[l] + zp, alpha, beta, Z, ucut);
        if (P.wall_mode == 1) v -= or_es_dphi(z_nodes[l] - (2.0 * P.H - zp), alpha, beta, Z, ucut);
        g.dzeta[l] = v;
    }
}

extern "C" {

// grid[c][l][j][i] += (1/2) (G(p; i, j, l) x tau_p)_c   — ADDS to grid (the force field of or_spread is already there)
void or_spread_curl(const or_params* P, int n, const double* pos, const double* tau, double beta, double* grid) {
    size_t plane = (size_t)P->nx * P->ny, field = plane * P->nz;
    double h = P->Lx / P->nx, alpha = 0.5 * P->w * h;
    double Z = or_es_norm(alpha, beta), ucut = or_es_dphi_cut(beta);
    std::vector<double> zn(P->nz);
    or_cheb_nodes(P->nz, P->H, zn.data());
    GradFootprint g;
    for (int p = 0; p < n; ++p) {
        grad_footprint(*P, beta, Z, ucut, zn.data(), pos + 3 * (size_t)p, g);
        const double* t = tau + 3 * (size_t)p;
        for (int l = 0; l < P->nz; ++l) {
            if (g.fp.zeta[l] == 0.0 && g.dzeta[l] == 0.0) continue;
            for (int b = 0; b < P->w; ++b) {
                int j = pmod(g.fp.j0 + b, P->ny);
                for (int a = 0; a < P->w; ++a) {
                    int i = pmod(g.fp.i0 + a, P->nx);
                    double Gx = g.dpx[a] * g.fp.py[b] * g.fp.zeta[l];
                    double Gy = g.fp.px[a] * g.dpy[b] * g.fp.zeta[l];
                    double Gz = g.fp.px[a] * g.fp.py[b] * g.dzeta[l];
                    size_t o = l * plane + (size_t)j * P->nx + i;
                    grid[0 * field + o] += 0.5 * (Gy * t[2] - Gz * t[1]);
                    grid[1 * field + o] += 0.5 * (Gz * t[0] - Gx * t[2]);
                    grid[2 * field + o] += 0.5 * (Gx * t[1] - Gy * t[0]);
                }
            }
        }
    }
}

// out[p] = (1/2) sum_{i,j,l} (u(i,j,l) x G(p; i, j, l)) h^2 (H/2) w_l,   u = grid[0..2]
void or_interp_curl(const or_params* P, int n, const double* pos, const double* grid, double beta, double* out) {
    size_t plane = (size_t)P->nx * P->ny, field = plane * P->nz;
    double h = P->Lx / P->nx, alpha = 0.5 * P->w * h;
    double Z = or_es_norm(alpha, beta), ucut = or_es_dphi_cut(beta);
    std::vector<double> zn(P->nz), wq(P->nz);
    or_cheb_nodes(P->nz, P->H, zn.data());
    or_cc_weights(P->nz, wq.data());
#pragma omp parallel
    {
        GradFootprint g;
#pragma omp for schedule(static)
        for (int p = 0; p < n; ++p) {
            grad_footprint(*P, beta, Z, ucut, zn.data(), pos + 3 * (size_t)p, g);
            double s[3] = {0, 0, 0};
            for (int l = 0; l < P->nz; ++l) {
                if (g.fp.zeta[l] == 0.0 && g.dzeta[l] == 0.0) continue;
                double wl = h * h * (0.5 * P->H) * wq[l];
                for (int b = 0; b < P->w; ++b) {
                    int j = pmod(g.fp.j0 + b, P->ny);
                    for (int a = 0; a < P->w; ++a) {
                        int i = pmod(g.fp.i0 + a, P->nx);
                        double Gx = g.dpx[a] * g.fp.py[b] * g.fp.zeta[l];
                        double Gy = g.fp.px[a] * g.dpy[b] * g.fp.zeta[l];
                        double Gz = g.fp.px[a] * g.fp.py[b] * g.dzeta[l];
                        size_t o = l * plane + (size_t)j * P->nx + i;
                        double u = grid[0 * field + o], v = grid[1 * field + o], w = grid[2 * field + o];
                        s[0] += 0.5 * (v * Gz - w * Gy) * wl;
                        s[1] += 0.5 * (w * Gx - u * Gz) * wl;
                        s[2] += 0.5 * (u * Gy - v * Gx) * wl;
                    }
                }
            }
            for (int c = 0; c < 3; ++c) out[3 * (size_t)p + c] = s[c];
        }
    }
}

// O2: unnormalised forward DFT in x,y of nplanes real planes [j][i] -> half spectrum [ny][nkx]
//   f^(n_x, n_y) = sum_{i,j} f(i,j) exp(-2 pi i (n_x i/nx + n_y j/ny)),  n_x = 0..nx/2, n_y = 0..ny-1
// written as the two nested 1-D sums (x then y).  Explicit O(n^2) per line.
void or_dft_xy_forward(int nx, int ny, long nplanes, const double* in, double* out_ri) {
    cd* out = reinterpret_cast<cd*>(out_ri);
    int nkx = nx / 2 + 1;
    std::vector<cd> twx(nx), twy(ny);
    for (int m = 0; m < nx; ++m) twx[m] = cd((double)cosl(-2 * PI_L * m / nx), (double)sinl(-2 * PI_L * m / nx));
    for (int m = 0; m < ny; ++m) twy[m] = cd((double)cosl(-2 * PI_L * m / ny), (double)sinl(-2 * PI_L * m / ny));
#pragma omp parallel
    {
        std::vector<cd> g((size_t)ny * nkx);
#pragma omp for schedule(dynamic, 1)
        for (long pl = 0; pl < nplanes; ++pl) {
            const double* f = in + (size_t)pl * nx * ny;
            for (int j = 0; j < ny; ++j)
                for (int kx = 0; kx < nkx; ++kx) {
                    cd s = 0;
                    for (int i = 0; i < nx; ++i) s += f[(size_t)j * nx + i] * twx[(size_t)((long)kx * i % nx)];
                    g[(size_t)j * nkx + kx] = s;
                }
            cd* o = out + (size_t)pl * ny * nkx;
            for (int ky = 0; ky < ny; ++ky)
                for (int kx = 0; kx < nkx; ++kx) {
                    cd s = 0;
                    for (int j = 0; j < ny; ++j) s += g[(size_t)j * nkx + kx] * twy[(size_t)((long)ky * j % ny)];
                    o[(size_t)ky * nkx + kx] = s;
                }
        }
    }
}

// O11: inverse DFT with Hermitian completion of the half spectrum and 1/(nx ny):
//   u(i,j) = (1/(nx ny)) sum_{n_x=0}^{nx-1} sum_{n_y} u^(n_x,n_y) exp(+2 pi i (n_x i/nx + n_y j/ny)),
//   with u^(nx-n_x, -n_y) = conj u^(n_x, n_y); real part.  (Equivalent to a C2R transform.)
void or_dft_xy_inverse(int nx, int ny, long nplanes, const double* in_ri, double* out) {
    const cd* in = reinterpret_cast<const cd*>(in_ri);
    int nkx = nx / 2 + 1;
    std::vector<cd> twx(nx), twy(ny);
    for (int m = 0; m < nx; ++m) twx[m] = cd((double)cosl(2 * PI_L * m / nx), (double)sinl(2 * PI_L * m / nx));
    for (int m = 0; m < ny; ++m) twy[m] = cd((double)cosl(2 * PI_L * m / ny), (double)sinl(2 * PI_L * m / ny));
#pragma omp parallel
    {
        std::vector<cd> g((size_t)ny * nkx);
#pragma omp for schedule(dynamic, 1)
        for (long pl = 0; pl < nplanes; ++pl) {
            const cd* uh = in + (size_t)pl * ny * nkx;
            for (int j = 0; j < ny; ++j)
                for (int kx = 0; kx < nkx; ++kx) {
                    cd s = 0;
                    for (int ky = 0; ky < ny; ++ky) s += uh[(size_t)ky * nkx + kx] * twy[(size_t)((long)ky * j % ny)];
                    g[(size_t)j * nkx + kx] = s;
                }
            double* u = out + (size_t)pl * nx * ny;
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    // n_x = 0 and (nx even) n_x = nx/2 appear once; 0 < n_x < nx/2 pairs with its conjugate
                    double s = g[(size_t)j * nkx].real();
                    for (int kx = 1; kx < nkx; ++kx) {
                        cd t = g[(size_t)j * nkx + kx] * twx[(size_t)((long)kx * i % nx)];
                        bool unpaired = (nx % 2 == 0 && kx == nx / 2);
                        s += unpaired ? t.real() : 2.0 * t.real();
                    }
                    u[(size_t)j * nx + i] = s / ((double)nx * ny);
                }
        }
    }
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// The oracle's own plain FFT (SURVEY.md §8(d) "CPU baseline": "its own plain recursive mixed-radix FFT, validated
// against its naive DFT").  It computes exactly the sums of or_dft_xy_forward / or_dft_xy_inverse (O2, O11), by the
// textbook Cooley-Tukey recursion on the smallest prime factor p of n (n = p m):
//   X[k + q m] = sum_{r<p} W_n^{r (k + q m)} Y_r[k],   Y_r = DFT_m of x[r], x[r+p], ...,   k < m, q < p,
// and the plain O(n^2) sum when n is prime.  No real-input trick, no blocking, out of place, twiddles from one table
// exp(sign 2 pi i j / n) evaluated in long double.  Pinned against the naive sums in tests/test_oracle_basics.py.
static int smallest_prime_factor(int n) {
    for (int p = 2; (long)p * p <= n; ++p) if (n % p == 0) return p;
    return n;
}

// DFT of the n numbers in[0], in[istride], ... -> out[0..n-1]; root[j * rstep] = exp(sign 2 pi i j / n), j < n
static void fft_plain(int n, const cd* in, long istride, cd* out, const cd* root, long rstep) {
    if (n == 1) { out[0] = in[0]; return; }
    const int p = smallest_prime_factor(n), m = n / p;
    if (p == n) {
        for (int k = 0; k < n; ++k) {
            cd s = 0;
            for (int j = 0; j < n; ++j) s += in[j * istride] * root[(long)((long)j * k % n) * rstep];
            out[k] = s;
        }
        return;
    }
    for (int r = 0; r < p; ++r) fft_plain(m, in + r * istride, istride * p, out + (long)r * m, root, rstep * p);
    cd tsmall[8];
    std::vector<cd> tlarge;
    cd* t = tsmall;
    if (p > 8) { tlarge.resize(p); t = tlarge.data(); }
    for (int k = 0; k < m; ++k) {
        for (int r = 0; r < p; ++r) t[r] = out[(long)r * m + k] * root[(long)r * k * rstep];              // W_n^{r k}, r k < n
        for (int q = 0; q < p; ++q) {
            cd s = 0;
            for (int r = 0; r < p; ++r) s += t[r] * root[(long)((r * q) % p) * m * rstep];                  // W_n^{r q m} = W_p^{r q}
            out[k + (long)q * m] = s;
        }
    }
}

static void root_table(int n, int sign, std::vector<cd>& root) {
    root.resize(n);
    for (int j = 0; j < n; ++j) root[j] = cd((double)cosl(2 * PI_L * j / n), (double)(sign * sinl(2 * PI_L * j / n)));
}

extern "C" {

// O2 through fft_plain: same definition as or_dft_xy_forward (x then y, unnormalised, half spectrum kept)
void or_fft_xy_forward(int nx, int ny, long nplanes, const double* in, double* out_ri) {
    cd* out = reinterpret_cast<cd*>(out_ri);
    const int nkx = nx / 2 + 1;
    std::vector<cd> rx, ry;
    root_table(nx, -1, rx); root_table(ny, -1, ry);
#pragma omp parallel
    {
        std::vector<cd> row(nx), spec(nx), g((size_t)ny * nkx), col(ny), cs(ny);
#pragma omp for schedule(dynamic, 1)
        for (long pl = 0; pl < nplanes; ++pl) {
            const double* f = in + (size_t)pl * nx * ny;
            for (int j = 0; j < ny; ++j) {
                for (int i = 0; i < nx; ++i) row[i] = cd(f[(size_t)j * nx + i], 0.0);
                fft_plain(nx, row.data(), 1, spec.data(), rx.data(), 1);
                for (int kx = 0; kx < nkx; ++kx) g[(size_t)j * nkx + kx] = spec[kx];
            }
            cd* o = out + (size_t)pl * ny * nkx;
            for (int kx = 0; kx < nkx; ++kx) {
                for (int j = 0; j < ny; ++j) col[j] = g[(size_t)j * nkx + kx];
                fft_plain(ny, col.data(), 1, cs.data(), ry.data(), 1);
                for (int ky = 0; ky < ny; ++ky) o[(size_t)ky * nkx + kx] = cs[ky];
            }
        }
    }
}

// O11 through fft_plain: inverse in y on the half spectrum, Hermitian completion of every x row
// (u^(nx - n_x) = conj u^(n_x) after the y sum), inverse in x, real part, 1/(nx ny)
void or_fft_xy_inverse(int nx, int ny, long nplanes, const double* in_ri, double* out) {
    const cd* in = reinterpret_cast<const cd*>(in_ri);
    const int nkx = nx / 2 + 1;
    std::vector<cd> rx, ry;
    root_table(nx, +1, rx); root_table(ny, +1, ry);
#pragma omp parallel
    {
        std::vector<cd> row(nx), res(nx), g((size_t)ny * nkx), col(ny), cs(ny);
#pragma omp for schedule(dynamic, 1)
        for (long pl = 0; pl < nplanes; ++pl) {
            const cd* uh = in + (size_t)pl * ny * nkx;
            for (int kx = 0; kx < nkx; ++kx) {
                for (int ky = 0; ky < ny; ++ky) col[ky] = uh[(size_t)ky * nkx + kx];
                fft_plain(ny, col.data(), 1, cs.data(), ry.data(), 1);
                for (int j = 0; j < ny; ++j) g[(size_t)j * nkx + kx] = cs[j];
            }
            double* u = out + (size_t)pl * nx * ny;
            for (int j = 0; j < ny; ++j) {
                for (int kx = 0; kx < nkx; ++kx) row[kx] = g[(size_t)j * nkx + kx];
                for (int kx = 1; kx < nkx; ++kx) if (nx - kx >= nkx) row[nx - kx] = std::conj(g[(size_t)j * nkx + kx]);
                fft_plain(nx, row.data(), 1, res.data(), rx.data(), 1);
                for (int i = 0; i < nx; ++i) u[(size_t)j * nx + i] = res[i].real() / ((double)nx * ny);
            }
        }
    }
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// Dense LU with partial pivoting, long double matrix (real), complex or real right-hand sides.
struct LU {
    int n;
    std::vector<ld> a;
    std::vector<int> piv;
    void factor(const std::vector<ld>& M, int n_) {
        n = n_; a = M; piv.resize(n);
        for (int c = 0; c < n; ++c) {
            int p = c; ld best = fabsl(a[(size_t)c * n + c]);
            for (int r = c + 1; r < n; ++r) if (fabsl(a[(size_t)r * n + c]) > best) { best = fabsl(a[(size_t)r * n + c]); p = r; }
            piv[c] = p;
            if (p != c) for (int k = 0; k < n; ++k) std::swap(a[(size_t)c * n + k], a[(size_t)p * n + k]);
            ld d = a[(size_t)c * n + c];
            for (int r = c + 1; r < n; ++r) {
                ld m = a[(size_t)r * n + c] / d;
                a[(size_t)r * n + c] = m;
                for (int k = c + 1; k < n; ++k) a[(size_t)r * n + k] -= m * a[(size_t)c * n + k];
            }
        }
    }
    void solve(std::vector<cld>& b) const {
        for (int c = 0; c < n; ++c) if (piv[c] != c) std::swap(b[c], b[piv[c]]);       // P b (full rows were swapped in factor)
        for (int c = 0; c < n; ++c) for (int r = c + 1; r < n; ++r) b[r] -= a[(size_t)r * n + c] * b[c];
        for (int r = n - 1; r >= 0; --r) { cld s = b[r]; for (int k = r + 1; k < n; ++k) s -= a[(size_t)r * n + k] * b[k]; b[r] = s / a[(size_t)r * n + r]; }
    }
};

// Dense complex solve (small systems: slit-channel 8x8), long double, partial pivoting, row equilibration.
static void dense_solve_c(std::vector<cld>& A, std::vector<cld>& b, int n) {
    for (int r = 0; r < n; ++r) {
        ld m = 0; for (int c = 0; c < n; ++c) m = std::max(m, std::abs(A[(size_t)r * n + c]));
        if (m > 0) { for (int c = 0; c < n; ++c) A[(size_t)r * n + c] /= m; b[r] /= m; }
    }
    for (int c = 0; c < n; ++c) {
        int p = c; ld best = std::abs(A[(size_t)c * n + c]);
        for (int r = c + 1; r < n; ++r) if (std::abs(A[(size_t)r * n + c]) > best) { best = std::abs(A[(size_t)r * n + c]); p = r; }
        if (p != c) { for (int k = 0; k < n; ++k) std::swap(A[(size_t)c * n + k], A[(size_t)p * n + k]); std::swap(b[c], b[p]); }
        for (int r = c + 1; r < n; ++r) {
            cld m = A[(size_t)r * n + c] / A[(size_t)c * n + c];
            for (int k = c; k < n; ++k) A[(size_t)r * n + k] -= m * A[(size_t)c * n + k];
            b[r] -= m * b[c];
        }
    }
    for (int r = n - 1; r >= 0; --r) { cld s = b[r]; for (int k = r + 1; k < n; ++k) s -= A[(size_t)r * n + k] * b[k]; b[r] = s / A[(size_t)r * n + r]; }
}

// Per-plan dense Chebyshev operators in long double.
struct ChebOps {
    int nz; ld H;
    std::vector<ld> A, S, D, D2, z;    // analysis [n][l], synthesis [l][n], derivative [n][m], D*D, nodes
    ChebOps(int nz_, double H_) : nz(nz_), H(H_) {
        int N = nz - 1;
        A.resize((size_t)nz * nz); S.resize((size_t)nz * nz); z.resize(nz);
        for (int n = 0; n < nz; ++n)
            for (int l = 0; l < nz; ++l) {
                ld cn = (n == 0 || n == N) ? 2 : 1, cl = (l == 0 || l == N) ? 2 : 1;
                A[(size_t)n * nz + l] = (2.0L / N) / (cn * cl) * cosl(PI_L * n * l / N);
                S[(size_t)l * nz + n] = cosl(PI_L * n * l / N);
            }
        for (int l = 0; l < nz; ++l) z[l] = (ld)(0.5 * H_ * (1.0 + cos(M_PI * l / (nz - 1))));   // the fp64 nodes
        cheb_diff_matrix_ld(nz, H, D);
        D2.assign((size_t)nz * nz, 0);
        for (int i = 0; i < nz; ++i) for (int k = 0; k < nz; ++k) { ld d = D[(size_t)i * nz + k]; if (d != 0) for (int j = 0; j < nz; ++j) D2[(size_t)i * nz + j] += d * D[(size_t)k * nz + j]; }
    }
    void analysis(const std::vector<cld>& nodal, std::vector<cld>& coef) const {
        coef.assign(nz, cld(0));
        for (int n = 0; n < nz; ++n) { cld s = 0; for (int l = 0; l < nz; ++l) s += A[(size_t)n * nz + l] * nodal[l]; coef[n] = s; }
    }
    void synthesis(const std::vector<cld>& coef, std::vector<cld>& nodal) const {
        nodal.assign(nz, cld(0));
        for (int l = 0; l < nz; ++l) { cld s = 0; for (int n = 0; n < nz; ++n) s += S[(size_t)l * nz + n] * coef[n]; nodal[l] = s; }
    }
    void diff(const std::vector<cld>& c, std::vector<cld>& d) const {
        d.assign(nz, cld(0));
        for (int n = 0; n < nz; ++n) { cld s = 0; for (int m = n + 1; m < nz; m += 2) s += D[(size_t)n * nz + m] * c[m]; d[n] = s; }
    }
    static cld at_top(const std::vector<cld>& c) { cld s = 0; for (size_t n = 0; n < c.size(); ++n) s += c[n]; return s; }             // z = H, xi = +1
    static cld at_bottom(const std::vector<cld>& c) { cld s = 0; for (size_t n = 0; n < c.size(); ++n) s += (n % 2 ? -c[n] : c[n]); return s; }  // z = 0
};

// The Chebyshev-tau BVP matrix of O5:  rows 0..nz-3: (D^2 - k^2 I);
// row nz-2: (d/dz + k) at z = H;  row nz-1: (d/dz - k) at z = 0   (eqs 15, 17, 18, 22, 24)
static void bvp_matrix(const ChebOps& C, ld k, std::vector<ld>& M) {
    int nz = C.nz;
    M.assign((size_t)nz * nz, 0);
    for (int n = 0; n < nz - 2; ++n) { for (int m = 0; m < nz; ++m) M[(size_t)n * nz + m] = C.D2[(size_t)n * nz + m]; M[(size_t)n * nz + n] -= k * k; }
    for (int m = 0; m < nz; ++m) {
        ld sH = 0, s0 = 0;
        for (int n = 0; n < nz; ++n) { sH += C.D[(size_t)n * nz + m]; s0 += (n % 2 ? -1 : 1) * C.D[(size_t)n * nz + m]; }
        M[(size_t)(nz - 2) * nz + m] = sH + k;
        M[(size_t)(nz - 1) * nz + m] = s0 - k * (m % 2 ? -1 : 1);
    }
}

// k = 0 matrix of O9: rows 0..nz-3: D^2; row nz-2: u(0) - l0 u'(0) (BW: l0 = 0: eq 52; slit: (A12));
// row nz-1: BW: u'(H) (eq 52); slit: u(H) + lH u'(H)  ((A12))
static void zero_mode_matrix(const ChebOps& C, int wall_mode, ld l0, ld lH, std::vector<ld>& M) {
    int nz = C.nz;
    M.assign((size_t)nz * nz, 0);
    for (int n = 0; n < nz - 2; ++n) for (int m = 0; m < nz; ++m) M[(size_t)n * nz + m] = C.D2[(size_t)n * nz + m];
    for (int m = 0; m < nz; ++m) {
        ld dH = 0, d0 = 0;                                                           // sum (D u)_n = u'(H), sum (-1)^n (D u)_n = u'(0)
        for (int n = 0; n < nz; ++n) { dH += C.D[(size_t)n * nz + m]; d0 += (n % 2 ? -1 : 1) * C.D[(size_t)n * nz + m]; }
        M[(size_t)(nz - 2) * nz + m] = (m % 2 ? -1 : 1) - l0 * d0;                   // sum (-1)^n u_n = u(z=0)
        if (wall_mode == 0) M[(size_t)(nz - 1) * nz + m] = dH;
        else M[(size_t)(nz - 1) * nz + m] = 1 + lH * dH;                             // sum u_n = u(z=H)
    }
}

extern "C" {

// Solve the DP BVP  (d^2/dz^2 - k^2) y = r,  (d/dz + k) y(H) = rho_H,  (d/dz - k) y(0) = rho_0  for one
// right-hand side given by Chebyshev coefficients r[0..nz-3] (complex, interleaved) — exposed for the pins.
void or_bvp_solve(int nz, double H, double k, const double* r_ri, const double* rhoH_ri, const double* rho0_ri, double* y_ri) {
    ChebOps C(nz, H);
    std::vector<ld> M; bvp_matrix(C, k, M);
    LU lu; lu.factor(M, nz);
    std::vector<cld> b(nz);
    for (int n = 0; n < nz - 2; ++n) b[n] = cld(r_ri[2 * n], r_ri[2 * n + 1]);
    b[nz - 2] = cld(rhoH_ri[0], rhoH_ri[1]); b[nz - 1] = cld(rho0_ri[0], rho0_ri[1]);
    lu.solve(b);
    for (int n = 0; n < nz; ++n) { y_ri[2 * n] = (double)b[n].real(); y_ri[2 * n + 1] = (double)b[n].imag(); }
}

}  // extern "C"

// O3-O10 for a set of retained wavenumbers.  Inputs: nodal-in-z spectra of the spread force field fh[3][nz][K] and
// (optional) torque field th, K columns, column q belonging to the wavenumber index pair (ix, iy); outputs: nodal-in-z
// spectra of u (uh) and, if wanted, of (1/2) curl u (wh), same layout.  ixs == NULL: the columns are the whole half
// spectrum in its natural order, K = ny * nkx, q = iy * nkx + ix (or_solve); else column q is mode (ixs[q], iys[q])
// (or_solve_modes: the same body on a list of modes, for full-size parity checks on sampled columns).
// If dump_coef != NULL it receives the Chebyshev coefficients of the total velocity [3][nz][K] (stage dump).
static void solve_columns(const or_params* P, long ncols, const int* ixs, const int* iys, const double* fh_ri, const double* th_ri,
                          double* uh_ri, double* wh_ri, double* dump_coef_ri) {
    const int nx = P->nx, ny = P->ny, nz = P->nz, nkx = nx / 2 + 1;
    const size_t K = (size_t)ncols, field = K * nz;
    const cd* fh = reinterpret_cast<const cd*>(fh_ri);
    const cd* th = reinterpret_cast<const cd*>(th_ri);
    cd* uh = reinterpret_cast<cd*>(uh_ri);
    cd* wh = reinterpret_cast<cd*>(wh_ri);
    cd* dump = reinterpret_cast<cd*>(dump_coef_ri);
    const ChebOps C(nz, P->H);
    const ld eta = P->eta, H = P->H;
    const cld I(0, 1);

#pragma omp parallel
    {
        std::vector<cld> nod(nz), fc[3], tc[3], dt[3], tmp, r(nz), p, dp, uc[3], ucorr[3], utot[3], ucoef[3], dcoef[3], om[3], omn;
        std::vector<ld> M;
        LU lu;
#pragma omp for schedule(dynamic, 64)
        for (long q = 0; q < (long)K; ++q) {
            const int iy = ixs ? iys[q] : (int)(q / nkx), ix = ixs ? ixs[q] : (int)(q % nkx);
            const int nyq = (iy <= ny / 2) ? iy : iy - ny;          // FFT order
            const ld kx = 2 * PI_L * ix / (ld)P->Lx, ky = 2 * PI_L * nyq / (ld)P->Ly;
            const ld k = sqrtl(kx * kx + ky * ky);                  // magnitude always uses the full values (G5)
            // component ("first-derivative") multipliers vanish on the unpaired Nyquist index
            const ld kxt = (nx % 2 == 0 && ix == nx / 2) ? 0 : kx;
            const ld kyt = (ny % 2 == 0 && iy == ny / 2) ? 0 : ky;

            // O3: Chebyshev coefficients of f^ (and t^)
            for (int c = 0; c < 3; ++c) {
                for (int l = 0; l < nz; ++l) nod[l] = (cld)fh[c * field + (size_t)l * K + q];
                C.analysis(nod, fc[c]);
                if (th) {
                    for (int l = 0; l < nz; ++l) nod[l] = (cld)th[c * field + (size_t)l * K + q];
                    C.analysis(nod, tc[c]);
                    C.diff(tc[c], dt[c]);
                }
            }
            // O4: f^ += (1/2) curl t^   (eq 7)
            if (th)
                for (int n = 0; n < nz; ++n) {
                    fc[0][n] += 0.5L * (I * kyt * tc[2][n] - dt[1][n]);
                    fc[1][n] += 0.5L * (dt[0][n] - I * kxt * tc[2][n]);
                    fc[2][n] += 0.5L * (I * kxt * tc[1][n] - I * kyt * tc[0][n]);
                }

            if (ix == 0 && iy == 0) {
                // O9: k = 0 column (eqs 47, 51, 52, (A12)); no DP/correction split
                // the unnormalised xy DFT of a uniform wall velocity U is nx ny U at k = 0 and nothing elsewhere (eqs 46, 52, (A12))
                zero_mode_matrix(C, P->wall_mode, P->wall_mode == 1 ? (ld)P->slip_0 : 0, P->wall_mode == 1 ? (ld)P->slip_H : 0, M);
                lu.factor(M, nz);
                for (int c = 0; c < 2; ++c) {
                    std::vector<cld> b(nz, cld(0));
                    for (int n = 0; n < nz - 2; ++n) b[n] = -fc[c][n] / eta;
                    b[nz - 2] = (ld)nx * ny * (ld)P->uwall_0[c];
                    if (P->wall_mode == 1) b[nz - 1] = (ld)nx * ny * (ld)P->uwall_H[c];
                    lu.solve(b);
                    ucoef[c] = b;
                }
                ucoef[2].assign(nz, cld(0));
                for (int c = 0; c < 3; ++c) C.synthesis(ucoef[c], utot[c]);
            } else {
                // O5: pressure BVP (eqs 15, 17)
                bvp_matrix(C, k, M);
                lu.factor(M, nz);
                C.diff(fc[2], tmp);
                for (int n = 0; n < nz - 2; ++n) r[n] = I * kxt * fc[0][n] + I * kyt * fc[1][n] + tmp[n];
                r[nz - 2] = 0; r[nz - 1] = 0;
                p = r; lu.solve(p);
                C.diff(p, dp);
                const cld pH = ChebOps::at_top(p), p0 = ChebOps::at_bottom(p);        // "direct summation", step 3
                // O6: velocity BVPs (eqs 18, 22, 24)
                const ld kc[2] = {kxt, kyt};
                for (int c = 0; c < 2; ++c) {
                    for (int n = 0; n < nz - 2; ++n) r[n] = (I * kc[c] * p[n] - fc[c][n]) / eta;
                    r[nz - 2] = -(I * kc[c] / (2 * k * eta)) * pH;
                    r[nz - 1] = +(I * kc[c] / (2 * k * eta)) * p0;
                    uc[c] = r; lu.solve(uc[c]);
                }
                for (int n = 0; n < nz - 2; ++n) r[n] = (dp[n] - fc[2][n]) / eta;
                r[nz - 2] = pH / (2 * eta);
                r[nz - 1] = p0 / (2 * eta);
                uc[2] = r; lu.solve(uc[2]);

                // O7: wall data (eq 27; (A3a-d)): a uniform wall velocity has no k != 0 component;
                //   u_0 = -u_DP(0) + l0 du_DP/dz(0), u_H = -u_DP(H) - lH du_DP/dz(H) for the tangential components, w unchanged;
                //   the wall derivatives "by Chebyshev differentiation and direct summation" (footnote 46)
                const ld l0 = P->wall_mode == 1 ? (ld)P->slip_0 : 0, lH = P->wall_mode == 1 ? (ld)P->slip_H : 0;
                cld u0[3], uH[3];
                for (int c = 0; c < 3; ++c) { u0[c] = -ChebOps::at_bottom(uc[c]); uH[c] = -ChebOps::at_top(uc[c]); }
                if (l0 != 0 || lH != 0)
                    for (int c = 0; c < 2; ++c) {
                        C.diff(uc[c], tmp);
                        u0[c] += l0 * ChebOps::at_bottom(tmp);
                        uH[c] -= lH * ChebOps::at_top(tmp);
                    }

                // O8: correction at the nodes
                for (int c = 0; c < 3; ++c) ucorr[c].assign(nz, cld(0));
                if (P->wall_mode == 0) {
                    // eqs 42-44
                    const cld Q = I * k * u0[2] + kxt * u0[0] + kyt * u0[1];
                    const cld Wc = k * u0[2] - I * kxt * u0[0] - I * kyt * u0[1];
                    for (int l = 0; l < nz; ++l) {
                        ld zl = C.z[l], E = expl(-k * zl);
                        ucorr[0][l] = -(kxt / k) * Q * zl * E + u0[0] * E;
                        ucorr[1][l] = -(kyt / k) * Q * zl * E + u0[1] * E;
                        ucorr[2][l] = Wc * zl * E + u0[2] * E;
                    }
                } else {
                    // App. A ((A5), (A6), (A8), (A10)) with slip lengths l0, lH, unknowns
                    //   x = [C0, D0~, Cx, Dx~, Cy, Dy~, Cz, Dz~],  D~ = D e^{kH}  (basis e^{-k(H-z)})
                    const ld e = expl(-k * H);
                    std::vector<cld> A8(64, cld(0)), b8(8, cld(0));
                    auto at = [&](int r_, int c_) -> cld& { return A8[(size_t)r_ * 8 + c_]; };
                    const ld kcs[2] = {kxt, kyt};
                    for (int c = 0; c < 2; ++c) {
                        // (A8a): (i k_c l0/(2 eta k)) C0 - (i k_c l0/(2 eta k)) D0 + (1 + k l0) C_c + (1 - k l0) D_c = u_0
                        at(2 * c, 0) = +(I * kcs[c] * l0) / (2 * eta * k);
                        at(2 * c, 1) = -(I * kcs[c] * l0 * e) / (2 * eta * k);
                        at(2 * c, 2 + 2 * c) = 1 + k * l0; at(2 * c, 3 + 2 * c) = (1 - k * l0) * e; b8[2 * c] = u0[c];
                        // (A8c): (i k_c H e^{-kH}/(2 eta k)) (k lH - lH/H - 1) C0 + (i k_c H e^{kH}/(2 eta k)) (k lH + lH/H + 1) D0
                        //        + e^{-kH} (1 - k lH) C_c + e^{kH} (1 + k lH) D_c = u_H
                        at(2 * c + 1, 0) = (I * kcs[c] * H * e) / (2 * eta * k) * (k * lH - lH / H - 1);
                        at(2 * c + 1, 1) = (I * kcs[c] * H) / (2 * eta * k) * (k * lH + lH / H + 1);
                        at(2 * c + 1, 2 + 2 * c) = e * (1 - k * lH); at(2 * c + 1, 3 + 2 * c) = 1 + k * lH; b8[2 * c + 1] = uH[c];
                    }
                    // (A8b): Cz + Dz = w_0
                    at(4, 6) = 1; at(4, 7) = e; b8[4] = u0[2];
                    // (A8d): (H e^{-kH}/(2 eta)) C0 + (H e^{kH}/(2 eta)) D0 + e^{-kH} Cz + e^{kH} Dz = w_H
                    at(5, 0) = H * e / (2 * eta); at(5, 1) = H / (2 * eta); at(5, 6) = e; at(5, 7) = 1; b8[5] = uH[2];
                    // (A10a): C0/(2 eta) + D0/(2 eta) + i kx (Cx + Dx) + i ky (Cy + Dy) - k Cz + k Dz = 0
                    at(6, 0) = 1 / (2 * eta); at(6, 1) = e / (2 * eta);
                    at(6, 2) = I * kxt; at(6, 3) = I * kxt * e; at(6, 4) = I * kyt; at(6, 5) = I * kyt * e;
                    at(6, 6) = -k; at(6, 7) = k * e;
                    // (A10b): e^{-kH} C0/(2 eta) + e^{kH} D0/(2 eta) + i kx (e^{-kH} Cx + e^{kH} Dx) + ... - k e^{-kH} Cz + k e^{kH} Dz = 0
                    at(7, 0) = e / (2 * eta); at(7, 1) = 1 / (2 * eta);
                    at(7, 2) = I * kxt * e; at(7, 3) = I * kxt; at(7, 4) = I * kyt * e; at(7, 5) = I * kyt;
                    at(7, 6) = -k * e; at(7, 7) = k;
                    dense_solve_c(A8, b8, 8);
                    const cld C0 = b8[0], D0 = b8[1];
                    for (int l = 0; l < nz; ++l) {
                        ld zl = C.z[l], Em = expl(-k * zl), Ep = expl(-k * (H - zl));
                        for (int c = 0; c < 2; ++c)     // (A5)
                            ucorr[c][l] = -(C0 * I * kcs[c] / (2 * eta * k)) * zl * Em + (D0 * I * kcs[c] / (2 * eta * k)) * zl * Ep
                                          + b8[2 + 2 * c] * Em + b8[3 + 2 * c] * Ep;
                        ucorr[2][l] = (C0 / (2 * eta)) * zl * Em + (D0 / (2 * eta)) * zl * Ep + b8[6] * Em + b8[7] * Ep;   // (A6)
                    }
                }
                // O10: total nodal values = synth(DP coefficients) + correction at the nodes (eq 28, step 6)
                for (int c = 0; c < 3; ++c) {
                    C.synthesis(uc[c], utot[c]);
                    for (int l = 0; l < nz; ++l) utot[c][l] += ucorr[c][l];
                }
            }
            for (int c = 0; c < 3; ++c)
                for (int l = 0; l < nz; ++l) uh[c * field + (size_t)l * K + q] = cd((double)utot[c][l].real(), (double)utot[c][l].imag());

            if (wh || dump) {
                // coefficients of the total, then omega^ = (1/2)(ik, d/dz) x u^ in coefficient space (eq 11; G12)
                for (int c = 0; c < 3; ++c) { C.analysis(utot[c], ucoef[c]); C.diff(ucoef[c], dcoef[c]); }
                if (dump)
                    for (int c = 0; c < 3; ++c)
                        for (int n = 0; n < nz; ++n) dump[c * field + (size_t)n * K + q] = cd((double)ucoef[c][n].real(), (double)ucoef[c][n].imag());
                if (wh) {
                    for (int c = 0; c < 3; ++c) om[c].assign(nz, cld(0));
                    for (int n = 0; n < nz; ++n) {
                        om[0][n] = 0.5L * (I * kyt * ucoef[2][n] - dcoef[1][n]);
                        om[1][n] = 0.5L * (dcoef[0][n] - I * kxt * ucoef[2][n]);
                        om[2][n] = 0.5L * (I * kxt * ucoef[1][n] - I * kyt * ucoef[0][n]);
                    }
                    for (int c = 0; c < 3; ++c) {
                        C.synthesis(om[c], omn);
                        for (int l = 0; l < nz; ++l) wh[c * field + (size_t)l * K + q] = cd((double)omn[l].real(), (double)omn[l].imag());
                    }
                }
            }
        }
    }
}

extern "C" {

// every retained wavenumber: fh, th, uh, wh, dump are half spectra [3][nz][ny][nkx]
void or_solve(const or_params* P, const double* fh_ri, const double* th_ri, double* uh_ri, double* wh_ri, double* dump_coef_ri) {
    solve_columns(P, (long)P->ny * (P->nx / 2 + 1), nullptr, nullptr, fh_ri, th_ri, uh_ri, wh_ri, dump_coef_ri);
}

// a list of wavenumbers (ix[q], iy[q]), q < nmodes: arrays [3][nz][nmodes]
void or_solve_modes(const or_params* P, long nmodes, const int* ix, const int* iy, const double* fh_ri, const double* th_ri,
                    double* uh_ri, double* wh_ri) {
    solve_columns(P, nmodes, ix, iy, fh_ri, th_ri, uh_ri, wh_ri, nullptr);
}

}  // extern "C"
