"""Pins for the oracle's building blocks: ES kernel, Chebyshev operators, xy DFT.

Each check compares the oracle against something other than itself: a library routine
(numpy.polynomial.chebyshev, numpy.fft, scipy.integrate), a closed form, or a value printed in the paper
(tests/golden/paper_tables.txt).
"""
import math
import os

import numpy as np
import pytest
from numpy.polynomial import chebyshev as npcheb
from scipy import integrate

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- ES kernel (eq 54)
@pytest.mark.parametrize("alpha,beta", [(2.0, 6 * 1.714), (1.5, 4 * 1.785), (3.0, 6 * 2.216)])
def test_es_phi_unit_integral_and_shape(alpha, beta):
    phi = lambda s: oracle.es_phi(s, alpha, beta)[0]
    val, _ = integrate.quad(phi, -alpha, alpha, epsabs=1e-13, epsrel=1e-13, limit=400)
    assert abs(val - 1.0) < 1e-9                       # normalisation Z
    assert phi(0.0) == pytest.approx(1.0 / oracle.es_norm(alpha, beta), rel=1e-14)   # exp(0)/Z at the centre
    assert phi(alpha) == pytest.approx(math.exp(-beta) * phi(0.0), rel=1e-12)        # edge value e^{-beta}/Z (G6)
    assert phi(1.0000001 * alpha) == 0.0 and phi(-1.0000001 * alpha) == 0.0          # compact support
    assert phi(0.3 * alpha) == phi(-0.3 * alpha)                                        # even
    # semicircle exponent at s = alpha*sqrt(3)/2 : sqrt(1 - 3/4) = 1/2
    assert phi(alpha * math.sqrt(3) / 2) == pytest.approx(math.exp(-beta / 2) * phi(0.0), rel=1e-10)


def _rh_monopole(w, beta):
    """Closed form for a tensor-product envelope in unbounded Stokes flow (DESIGN.md pin P1):
    1/(6 pi eta R_h) = (2/(3 eta)) int_0^inf g(t)^3 dt,  g(t) = (1/pi) int_0^inf |phi^(q)|^2 exp(-q^2 t) dq."""
    alpha = w / 2.0                                    # h = 1
    xs, ws = np.polynomial.legendre.leggauss(200)
    s = alpha * xs
    ph = oracle.es_phi(s, alpha, beta) * alpha * ws    # quadrature of phi(s) ds
    q = np.linspace(0.0, 40.0, 8001)
    phat = (ph[None, :] * np.cos(q[:, None] * s[None, :])).sum(axis=1)
    p2 = phat ** 2

    def g(t):
        return integrate.simpson(p2 * np.exp(-q * q * t), x=q) / math.pi

    # t = tan^2-like map to [0, inf): t = u/(1-u)
    us, wu = np.polynomial.legendre.leggauss(400)
    u = 0.5 * (us + 1.0)
    t = u / (1.0 - u)
    integ = sum(0.5 * wi * g(ti) ** 3 / (1.0 - ui) ** 2 for wi, ti, ui in zip(wu, t, u))
    return 1.0 / (6.0 * math.pi * (2.0 / 3.0) * integ)


def _rh_dipole(w, beta):
    """R_h^D = (3/(4 pi))^(1/3) / int phi_D(s)^2 ds  (DESIGN.md pin P1)."""
    alpha = w / 2.0
    val, _ = integrate.quad(lambda s: oracle.es_phi(s, alpha, beta)[0] ** 2, -alpha, alpha, epsabs=1e-13, limit=400)
    return (3.0 / (4.0 * math.pi)) ** (1.0 / 3.0) / val


def _paper_table():
    rows = []
    with open(os.path.join(GOLD, "paper_tables.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                kind, w, bw, rh = line.split()
                rows.append((kind, int(w), float(bw), float(rh)))
    return rows


@pytest.mark.parametrize("kind,w,bw,rh", _paper_table())
def test_hydrodynamic_radius_matches_paper_tables(kind, w, bw, rh):
    """Tables I-II and PAPER.md:719: R_h/h for the printed (m, beta/m) to <= 1 %."""
    got = _rh_monopole(w, bw * w) if kind == "M" else _rh_dipole(w, bw * w)
    assert got == pytest.approx(rh, rel=0.01), (kind, w, bw, got)


def test_gaussian_limit_of_radius_formulas():
    """The two closed forms reduce to the paper's Gaussian relations g_M = R_h/sqrt(pi), g_D = R_h/(6 sqrt(pi))^(1/3)
    (eq 8) — analytic check of the pin itself, no oracle involved."""
    sig = 0.7
    # monopole: g(t) = 1/(2 sqrt(pi (sig^2 + t))), int g^3 = 1/(4 pi^1.5 sig)
    integ = 1.0 / (4.0 * math.pi ** 1.5 * sig)
    assert 1.0 / (6 * math.pi * (2 / 3) * integ) == pytest.approx(math.sqrt(math.pi) * sig, rel=1e-14)
    # dipole: int phi^2 = 1/(2 sqrt(pi) sig)
    rh = (3 / (4 * math.pi)) ** (1 / 3) * 2 * math.sqrt(math.pi) * sig
    assert rh == pytest.approx((6 * math.sqrt(math.pi)) ** (1 / 3) * sig, rel=1e-14)


# ---------------------------------------------------------------- Chebyshev pieces
@pytest.mark.parametrize("nz", [8, 19, 32, 48])
def test_cheb_nodes_and_transforms(nz):
    H = 7.3
    z = oracle.cheb_nodes(nz, H)
    assert z[0] == pytest.approx(H) and abs(z[-1]) < 1e-15 and np.all(np.diff(z) < 0)
    xi = 2 * z / H - 1
    rng = np.random.default_rng(nz)
    c = rng.standard_normal(nz)
    vals = npcheb.chebval(xi, c)                      # library evaluation of sum c_n T_n(xi)
    A = oracle.cheb_analysis_matrix(nz)
    S = oracle.cheb_synthesis_matrix(nz)
    assert np.allclose(A @ vals, c, atol=1e-13)       # analysis recovers the coefficients
    assert np.allclose(S @ c, vals, atol=1e-13)       # synthesis evaluates them
    assert np.allclose(A @ S, np.eye(nz), atol=1e-13)


@pytest.mark.parametrize("nz", [8, 32, 48])
def test_cheb_diff_matrix_against_chebder(nz):
    H = 5.0
    D = oracle.cheb_diff_matrix(nz, H)
    rng = np.random.default_rng(7)
    c = rng.standard_normal(nz)
    d = np.zeros(nz)
    d[: nz - 1] = npcheb.chebder(c) * (2.0 / H)       # d/dz = (2/H) d/dxi
    assert np.allclose(D @ c, d, rtol=1e-13, atol=1e-12)
    # the recurrence stated in SURVEY.md §8(c) gives the same thing
    r = np.zeros(nz + 2)
    for n in range(nz - 2, -1, -1):
        r[n] = r[n + 2] + 2 * (n + 1) * c[n + 1]
    r[0] *= 0.5
    assert np.allclose(D @ c, r[:nz] * (2.0 / H), rtol=1e-13, atol=1e-12)


@pytest.mark.parametrize("nz", [9, 32, 48])
def test_clenshaw_curtis_weights(nz):
    w = oracle.cc_weights(nz)
    assert w.sum() == pytest.approx(2.0, abs=1e-14)
    xi = np.cos(np.pi * np.arange(nz) / (nz - 1))
    for deg in range(0, nz):                          # exact for every polynomial of degree < nz
        exact = 0.0 if deg % 2 else 2.0 / (deg + 1)
        assert (w * xi ** deg).sum() == pytest.approx(exact, abs=1e-12)
    # a smooth non-polynomial: int_{-1}^{1} exp(xi) dxi
    if nz >= 16:
        assert (w * np.exp(xi)).sum() == pytest.approx(math.e - 1 / math.e, abs=1e-13)


# ---------------------------------------------------------------- xy DFT (O2, O11)
@pytest.mark.parametrize("nx,ny", [(8, 6), (12, 12), (9, 10), (10, 7)])
def test_dft_forward_is_rfft2_and_literal_double_sum(nx, ny):
    rng = np.random.default_rng(nx * 100 + ny)
    f = rng.standard_normal((3, ny, nx))
    got = oracle.dft_xy_forward(f, "naive")
    assert np.allclose(got, np.fft.rfft2(f, axes=(-2, -1)), atol=1e-12)
    # literal definition on plane 0
    i = np.arange(nx)[None, :]
    j = np.arange(ny)[:, None]
    for kx in range(nx // 2 + 1):
        for ky in range(ny):
            s = (f[0] * np.exp(-2j * np.pi * (kx * i / nx + ky * j / ny))).sum()
            assert abs(s - got[0, ky, kx]) < 1e-12
    assert np.allclose(oracle.dft_xy_forward(f, "fft"), got, atol=1e-12)
    assert np.allclose(oracle.dft_xy_forward(f, "numpy"), got, atol=1e-12)


@pytest.mark.parametrize("nx,ny", [(8, 6), (12, 12), (9, 10)])
def test_dft_inverse_roundtrip_and_irfft2(nx, ny):
    rng = np.random.default_rng(3)
    f = rng.standard_normal((2, ny, nx))
    spec = np.fft.rfft2(f, axes=(-2, -1))
    assert np.allclose(oracle.dft_xy_inverse(spec, nx, "naive"), f, atol=1e-13)
    assert np.allclose(oracle.dft_xy_inverse(spec, nx, "fft"), f, atol=1e-13)
    assert np.allclose(oracle.dft_xy_inverse(spec, nx, "numpy"), f, atol=1e-13)
    # full-spectrum definition with Hermitian completion
    full = np.fft.fft2(f, axes=(-2, -1))
    i = np.arange(nx)[None, :]
    j = np.arange(ny)[:, None]
    u00 = sum(full[0, ky, kx] * np.exp(2j * np.pi * (kx * 3 / nx + ky * 2 / ny)) for kx in range(nx) for ky in range(ny)) / (nx * ny)
    assert abs(u00.real - oracle.dft_xy_inverse(spec, nx, "naive")[0, 2, 3]) < 1e-13


@pytest.mark.parametrize("nx,ny", [(48, 48), (192, 192), (1080, 1080), (50, 28), (34, 22)])
def test_own_plain_fft_equals_the_naive_dft_sums(nx, ny):
    """The oracle's own recursive mixed-radix FFT (dft="fft", used where the O(n^2) sums do not finish) against its explicit
    DFT sums at the grid sizes of configs 1-3 (48, 192, 1080: SURVEY.md §8(d) "validated against its naive DFT to 1e-13 on
    configs 1-3") and at sizes with prime factors 7, 11, 17 (the prime-length branch); numpy.fft only as a third opinion."""
    rng = np.random.default_rng(nx + ny)
    f = rng.standard_normal((1, ny, nx))
    naive = oracle.dft_xy_forward(f, "naive")
    own = oracle.dft_xy_forward(f, "fft")
    scale = np.abs(naive).max()
    assert np.abs(own - naive).max() < 1e-13 * scale * max(1.0, np.log2(nx * ny) / 8)
    assert np.abs(oracle.dft_xy_forward(f, "numpy") - own).max() < 1e-13 * scale * max(1.0, np.log2(nx * ny) / 8)
    spec = naive * (rng.standard_normal(naive.shape) + 0.5)          # a generic Hermitian-completable half spectrum
    b_naive = oracle.dft_xy_inverse(spec, nx, "naive")
    b_own = oracle.dft_xy_inverse(spec, nx, "fft")
    assert np.abs(b_own - b_naive).max() < 1e-13 * np.abs(b_naive).max() * max(1.0, np.log2(nx * ny) / 8)
    # the imaginary parts of the kx = 0 and kx = nx/2 columns are what Hermitian completion must treat consistently
    assert np.abs(oracle.dft_xy_inverse(spec, nx, "numpy") - b_own).max() < 1e-12 * np.abs(b_naive).max()
