"""Pins for the oracle's per-wavenumber solve (O3-O10): DP boundary-value problems, wall corrections, k = 0.

Nothing here re-types the oracle's formulas.  The checks are: free-space Green's-function integrals, closed-form
homogeneous solutions, manufactured Stokes solutions (a divergence-free u vanishing on the wall(s) plus a
pressure, f computed from eq 4 symbolically with sympy), invariance under moving the artificial top boundary
(the Dirichlet-to-Neumann maps of eqs 17, 22, 24 make it transparent), the slit -> single wall limit, and the PDE
residuals of the output (no-slip, continuity, vorticity equation) via numpy's Chebyshev calculus.

The method needs a force density whose z-component is continuous across the computational boundaries (PAPER.md:125,
142: "p_DP is continuously differentiable across ..."; the image construction eq 9 guarantees it), so every test
source has f_z = 0 at z = 0 and z = H; f_x, f_y may be non-zero there.
"""
import math
from types import SimpleNamespace

import numpy as np
import pytest
import sympy as sp
from numpy.polynomial import chebyshev as npcheb
from scipy import integrate

import oracle

BW, SC = 0, 1
Z = sp.symbols("z", real=True)


def make_prob(wall_mode, H, nz, L=5.0, nxy=4, eta=1.3):
    return SimpleNamespace(wall_mode=wall_mode, Lx=L, Ly=L, H=H, nx=nxy, ny=nxy, nz=nz, w=6, beta_M=10.0, beta_D=12.0, eta=eta)


def wavenumbers(prob):
    nkx = prob.nx // 2 + 1
    kx = 2 * np.pi * np.arange(nkx) / prob.Lx
    ny = prob.ny
    ky = 2 * np.pi * np.where(np.arange(ny) <= ny // 2, np.arange(ny), np.arange(ny) - ny) / prob.Ly
    return kx, ky


def is_nyquist(prob, ix, iy):
    return (prob.nx % 2 == 0 and ix == prob.nx // 2) or (prob.ny % 2 == 0 and iy == prob.ny // 2)


class Fn:
    """A sympy expression in z with exact derivatives, evaluated with numpy."""

    def __init__(self, expr):
        self.expr = sp.sympify(expr)

    def d(self, m=1):
        return Fn(sp.diff(self.expr, Z, m))

    def __call__(self, z):
        z = np.asarray(z, dtype=float)
        return np.broadcast_to(np.asarray(sp.lambdify(Z, self.expr, "numpy")(z), dtype=float), z.shape).copy()


# ------------------------------------------------------------------------------------------------ BVP alone
@pytest.mark.parametrize("k", [0.3, 2.0, 6.0])
def test_bvp_matches_free_space_green_function(k):
    """(d2/dz2 - k^2) y = g on the line has y(z) = -(1/2k) int exp(-k|z-z'|) g(z') dz'; restricted to [0,H] it obeys
    the DtN conditions of eq 17.  Spectral convergence in nz."""
    H, nz, zc, sig = 8.0, 64, 3.7, 0.5
    g = lambda z: np.exp(-(z - zc) ** 2 / (2 * sig ** 2))
    z = oracle.cheb_nodes(nz, H)
    A = oracle.cheb_analysis_matrix(nz)
    S = oracle.cheb_synthesis_matrix(nz)
    r = (A @ g(z))[: nz - 2]
    y = S @ oracle.bvp_solve(nz, H, k, r)
    lo, hi = zc - 12 * sig, zc + 12 * sig
    q = lambda f, a, b: integrate.quad(f, a, b, epsabs=1e-14, epsrel=1e-13, points=[zc] if a < zc < b else None)[0]
    exact = np.array([-(1 / (2 * k)) * (q(lambda s: math.exp(-k * (zz - s)) * g(s), lo, zz) + q(lambda s: math.exp(-k * (s - zz)) * g(s), zz, hi))
                      for zz in z])
    assert np.max(np.abs(y.real - exact)) < 2e-8 * np.max(np.abs(exact))
    assert np.max(np.abs(y.imag)) == 0.0


def test_bvp_homogeneous_solution_with_boundary_data():
    """r = 0: y = (rho_H/2k) e^{k(z-H)} - (rho_0/2k) e^{-kz} satisfies (dz+k) y(H) = rho_H, (dz-k) y(0) = rho_0."""
    H, nz, k = 3.0, 40, 1.7
    rhoH, rho0 = 0.8 - 0.3j, -0.2 + 1.1j
    y = oracle.cheb_synthesis_matrix(nz) @ oracle.bvp_solve(nz, H, k, np.zeros(nz - 2), rhoH, rho0)
    z = oracle.cheb_nodes(nz, H)
    exact = rhoH / (2 * k) * np.exp(k * (z - H)) - rho0 / (2 * k) * np.exp(-k * z)
    assert np.max(np.abs(y - exact)) < 1e-12


# ------------------------------------------------------------------------------------------------ manufactured Stokes
def _manufactured(prob, W, Psi, Pr, tq=None):
    """Build f^ (nodal in z, all retained modes) from u^ = (i k/k^2) W' + (-ky, kx) Psi, w^ = W, pressure Pr via eq 4:
    f = -eta (dz^2 - k^2) u + (ik, dz) p.  Returns fh, th, exact u nodal, exact (1/2) curl u nodal."""
    nz, H, eta = prob.nz, prob.H, prob.eta
    z = oracle.cheb_nodes(nz, H)
    kxs, kys = wavenumbers(prob)
    shape = (3, nz, prob.ny, prob.nx // 2 + 1)
    fh = np.zeros(shape, complex); uex = np.zeros(shape, complex); omex = np.zeros(shape, complex)
    th = np.zeros(shape, complex) if tq is not None else None
    W0, W1, W2, W3 = W(z), W.d(1)(z), W.d(2)(z), W.d(3)(z)
    P0, P1, S0, S1, S2 = Pr(z), Pr.d(1)(z), Psi(z), Psi.d(1)(z), Psi.d(2)(z)
    tc = (0.3, -1.1j, 0.6 + 0.4j)
    for iy, ky in enumerate(kys):
        for ix, kx in enumerate(kxs):
            if (ix == 0 and iy == 0) or is_nyquist(prob, ix, iy):
                continue
            k2 = kx * kx + ky * ky
            amp = (0.7 + 0.2j) * (1 + 0.1 * ix - 0.05 * iy)
            u = amp * ((1j * kx / k2) * W1 - ky * S0)
            v = amp * ((1j * ky / k2) * W1 + kx * S0)
            w = amp * W0
            p = amp * P0
            lap_u = amp * ((1j * kx / k2) * W3 - ky * S2) - k2 * u
            lap_v = amp * ((1j * ky / k2) * W3 + kx * S2) - k2 * v
            lap_w = amp * W2 - k2 * w
            f = np.array([-eta * lap_u + 1j * kx * p, -eta * lap_v + 1j * ky * p, -eta * lap_w + amp * P1])
            uz = amp * ((1j * kx / k2) * W2 - ky * S1)
            vz = amp * ((1j * ky / k2) * W2 + kx * S1)
            om = 0.5 * np.array([1j * ky * w - vz, uz - 1j * kx * w, 1j * kx * v - 1j * ky * u])
            if tq is not None:
                t = np.array([c * amp * T(z) for c, T in zip(tc, tq)])
                tz = np.array([c * amp * T.d(1)(z) for c, T in zip(tc, tq)])
                curl_t = np.array([1j * ky * t[2] - tz[1], tz[0] - 1j * kx * t[2], 1j * kx * t[1] - 1j * ky * t[0]])
                f = f - 0.5 * curl_t                      # so that f + (1/2) curl t is the same total force density (eq 7)
                th[:, :, iy, ix] = t
            fh[:, :, iy, ix] = f
            uex[:, :, iy, ix] = [u, v, w]
            omex[:, :, iy, ix] = om
    return fh, th, uex, omex


def test_slit_manufactured_solution_forces_torques_and_curl():
    """Slit channel: a divergence-free u vanishing on both walls with a pressure is THE solution for its own f
    (eqs 4-6, App. A).  f_x, f_y do not vanish at the walls and the DP solution is far from no-slip, so the 8x8
    correction of App. A does real work.  Also pins O4 (torque curl, eq 7) and O10 (eq 11).
    The pressure is chosen with eta W'' = P' on the walls so that f_z is continuous there (module docstring)."""
    H = 3.0
    prob = make_prob(SC, H, nz=44)
    Wx = sp.sin(sp.pi * Z / H) ** 2 * (1 + 0.3 * Z)
    a0 = prob.eta * sp.diff(Wx, Z, 2).subs(Z, 0)
    aH = prob.eta * sp.diff(Wx, Z, 2).subs(Z, H)
    W = Fn(Wx)
    Psi = Fn(sp.sin(sp.pi * Z / H) * sp.exp(0.2 * Z))
    Pr = Fn(sp.cos(sp.pi * Z / H) * 0.8 + sp.cos(2 * sp.pi * Z / H) + a0 * (Z - Z ** 2 / (2 * H)) + aH * Z ** 2 / (2 * H))
    # the torque field's curl must not add a z-force on the walls either: its z-curl involves only t_x, t_y (no dz),
    # which are taken to vanish on the walls
    tq = [Fn(sp.sin(sp.pi * Z / H) * sp.cos(0.7 * Z)), Fn(sp.sin(sp.pi * Z / H) * sp.exp(-0.3 * Z)), Fn(1 + sp.sin(Z))]
    scale = None
    for torques in (None, tq):
        fh, th, uex, omex = _manufactured(prob, W, Psi, Pr, torques)
        assert np.max(np.abs(fh[2, [0, -1]])) < 1e-12 and np.max(np.abs(fh[0, [0, -1]])) > 0.1
        uh, wh, _ = oracle.solve(prob, fh, th, want_omega=True)
        scale = np.max(np.abs(uex))
        assert np.max(np.abs(uh - uex)) < 1e-10 * scale
        assert np.max(np.abs(wh - omex)) < 1e-8 * np.max(np.abs(omex))
    assert scale > 0.1


@pytest.mark.parametrize("wall_mode", [BW, SC])
def test_compact_manufactured_solution_both_geometries(wall_mode):
    """A compactly supported (to 1e-14) divergence-free u with compact pressure solves the bottom-wall AND the slit
    problem for its own f: pins the DP pressure/velocity solves (eqs 15-24) in both modes; correction ~ 0."""
    H, sig, zc = 8.0, 0.45, 3.9
    prob = make_prob(wall_mode, H, nz=72)
    G = sp.exp(-(Z - zc) ** 2 / (2 * sig ** 2))
    fh, th, uex, omex = _manufactured(prob, Fn(G), Fn(G * (1 + 0.1 * Z)), Fn(G * (0.3 + Z)))
    uh, wh, _ = oracle.solve(prob, fh, None, want_omega=True)
    assert np.max(np.abs(uh - uex)) < 1e-9 * np.max(np.abs(uex))
    assert np.max(np.abs(wh - omex)) < 1e-7 * np.max(np.abs(omex))


@pytest.mark.parametrize("wall_mode", [BW, SC])
def test_zero_mode_manufactured(wall_mode):
    """k = 0 (eqs 47, 51, 52; (A12)): u'' = -f/eta, u(0) = 0 and u'(H) = 0 (BW) / u(H) = 0 (slit), w = 0.
    With torques the k = 0 force is f - (1/2) dz t_y, f + (1/2) dz t_x (eq 7)."""
    H = 2.5
    prob = make_prob(wall_mode, H, nz=36)
    z = oracle.cheb_nodes(prob.nz, H)
    if wall_mode == BW:
        U = [Fn(sp.sin(sp.pi * Z / (2 * H))), Fn(Z * (2 * H - Z) * 0.3)]
    else:
        U = [Fn(sp.sin(sp.pi * Z / H) * (1 + Z)), Fn(Z * (H - Z) * sp.exp(0.3 * Z))]
    shape = (3, prob.nz, prob.ny, prob.nx // 2 + 1)
    fh = np.zeros(shape, complex); th = np.zeros(shape, complex)
    ty, tx = Fn(sp.cos(Z)), Fn(Z ** 2)
    amp = 1.0 + 0.5j
    # total force must be -eta U'':  f_x - (1/2) ty' = -eta Ux''  ,  f_y + (1/2) tx' = -eta Uy''
    fh[0, :, 0, 0] = (-prob.eta * U[0].d(2)(z) + 0.5 * ty.d(1)(z)) * amp
    fh[1, :, 0, 0] = (-prob.eta * U[1].d(2)(z) - 0.5 * tx.d(1)(z)) * amp
    fh[2, :, 0, 0] = np.cos(z)                          # any f_z: w(k=0) = 0 regardless (eq 47)
    th[0, :, 0, 0] = tx(z) * amp; th[1, :, 0, 0] = ty(z) * amp; th[2, :, 0, 0] = np.sin(z)
    uh, wh, _ = oracle.solve(prob, fh, th, want_omega=True)
    for c in range(2):
        assert np.max(np.abs(uh[c, :, 0, 0] - U[c](z) * amp)) < 1e-12
    assert np.max(np.abs(uh[2, :, 0, 0])) == 0.0
    assert np.max(np.abs(wh[0, :, 0, 0] - (-0.5) * U[1].d(1)(z) * amp)) < 1e-11
    assert np.max(np.abs(wh[1, :, 0, 0] - (+0.5) * U[0].d(1)(z) * amp)) < 1e-11
    assert np.max(np.abs(wh[2, :, 0, 0])) == 0.0


# ------------------------------------------------------------------------------------------------ generic sources
def _wall_source(prob, zs, both_walls=False, seed=11):
    """Smooth force density concentrated within ~zs of z = 0 (and of z = H if both_walls), vanishing ON the wall(s) with
    non-zero slope (like the image-folded particle sources) and, for the bottom wall, vanishing near z = H."""
    z = oracle.cheb_nodes(prob.nz, prob.H)
    shape = (3, prob.nz, prob.ny, prob.nx // 2 + 1)
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((3,) + shape[2:]) + 1j * rng.standard_normal((3,) + shape[2:])
    prof = z * np.exp(-(z / zs) ** 2) * (1 + 0.4 * z)
    if both_walls:
        prof = prof + 0.7 * (prob.H - z) * np.exp(-((prob.H - z) / (0.8 * zs)) ** 2)
    return a[:, None, :, :] * prof[None, :, None, None]


def _interp_z(prob, nodal, zq):
    """Evaluate the Chebyshev interpolant of nodal values (axis 0 = l) at heights zq, via numpy's vander solve."""
    z = oracle.cheb_nodes(prob.nz, prob.H)
    V = npcheb.chebvander(2 * z / prob.H - 1, prob.nz - 1)
    c = np.linalg.solve(V, nodal.reshape(prob.nz, -1))
    return (npcheb.chebvander(2 * zq / prob.H - 1, prob.nz - 1) @ c).reshape((len(zq),) + nodal.shape[1:])


@pytest.mark.parametrize("wall_mode", [BW, SC])
def test_output_satisfies_stokes_equations_and_no_slip(wall_mode):
    """For a generic source the output must satisfy: u = 0 on the wall(s) (eq 6); continuity (eq 5); and the curl of
    eq 4, eta (dz^2 - k^2) curl u = -curl f (pressure eliminated).  Checked with numpy's Chebyshev calculus."""
    H, nz = 6.0, 72
    prob = make_prob(wall_mode, H, nz, L=6.0)
    fh = _wall_source(prob, 1.1, both_walls=(wall_mode == SC))
    uh, wh, _ = oracle.solve(prob, fh, None, want_omega=True)
    z = oracle.cheb_nodes(nz, H)
    V = npcheb.chebvander(2 * z / H - 1, nz - 1)
    kxs, kys = wavenumbers(prob)
    umax = np.max(np.abs(uh))
    assert np.max(np.abs(uh[:, -1])) < 1e-12 * umax                      # z = 0 is node l = nz-1
    if wall_mode == SC:
        assert np.max(np.abs(uh[:, 0])) < 1e-12 * umax                   # z = H is node l = 0

    def dz(nod, m=1):
        return npcheb.chebval(2 * z / H - 1, npcheb.chebder(np.linalg.solve(V, nod), m)) * (2 / H) ** m

    checked = 0
    for iy, ky in enumerate(kys):
        for ix, kx in enumerate(kxs):
            if (ix == 0 and iy == 0) or is_nyquist(prob, ix, iy):
                continue
            k2 = kx * kx + ky * ky
            u, v, w = uh[0, :, iy, ix], uh[1, :, iy, ix], uh[2, :, iy, ix]
            f = fh[:, :, iy, ix]
            div = 1j * kx * u + 1j * ky * v + dz(w)
            assert np.max(np.abs(div)) < 1e-8 * np.max(np.abs(dz(w)))
            om2 = 2 * wh[:, :, iy, ix]                                   # curl u
            curl_f = np.array([1j * ky * f[2] - dz(f[1]), dz(f[0]) - 1j * kx * f[2], 1j * kx * f[1] - 1j * ky * f[0]])
            for c in range(3):
                res = prob.eta * (dz(om2[c], 2) - k2 * om2[c]) + curl_f[c]
                assert np.max(np.abs(res)) < 1e-6 * np.max(np.abs(curl_f)), (ix, iy, c)
            checked += 1
    assert checked >= 5


def test_bottom_wall_result_is_independent_of_the_artificial_top():
    """Bottom wall: z = H is not physical; the DtN conditions (eqs 17, 22, 24) make it transparent, so
    the same near-wall source solved with H = 5 and H = 9 must give the same u on [0, 5].  At small k the pressure and
    velocity are far from zero at z = 5, so the p(H) terms of eqs 22, 24 are exercised with their signs."""
    probA = make_prob(BW, 5.0, 64, L=20.0)
    probB = make_prob(BW, 9.0, 96, L=20.0)
    zq = np.linspace(0.0, 5.0, 23)
    outs = []
    for prob in (probA, probB):
        z = oracle.cheb_nodes(prob.nz, prob.H)
        shape = (3, prob.nz, prob.ny, prob.nx // 2 + 1)
        rng = np.random.default_rng(5)
        a = rng.standard_normal((3,) + shape[2:]) + 1j * rng.standard_normal((3,) + shape[2:])
        prof = z * np.exp(-((z - 0.8) / 0.7) ** 2)         # 0 on the wall, < 1e-15 beyond z = 5
        fh = a[:, None] * prof[None, :, None, None]
        uh, _, _ = oracle.solve(prob, fh, None)
        outs.append(np.stack([_interp_z(prob, uh[c], zq) for c in range(3)]))
    scale = np.max(np.abs(outs[0]))
    assert np.max(np.abs(outs[0][:, -1])) > 1e-2 * scale   # the field is NOT small at the truncation height
    assert np.max(np.abs(outs[0] - outs[1])) < 1e-8 * scale


def test_slit_tends_to_bottom_wall_when_the_top_wall_recedes():
    """P8 / PAPER.md:531: for k H >> 1 the top wall's influence on a near-bottom source vanishes: at height z it is
    O(e^{-k(2H - z)}), so the two solutions are compared near the bottom wall, where the source and the flow are."""
    L = 3.0                                                # k_min = 2.09: e^{-2 k H} = 3e-15 at H = 8
    probS = make_prob(SC, 8.0, 96, L=L)
    probB = make_prob(BW, 8.0, 96, L=L)
    fh = _wall_source(probS, 0.9, seed=6)
    fh[:, :, 0, 0] = 0                                      # k = 0 differs by construction (eq 52 vs (A12))
    uS, _, _ = oracle.solve(probS, fh, None)
    uB, _, _ = oracle.solve(probB, fh, None)
    lower = oracle.cheb_nodes(96, 8.0) <= 1.2      # measured prefactor of e^{-k(2H-z)} is ~5e2 (polynomial in kH)
    assert np.max(np.abs(uS - uB)[:, lower]) < 1e-9 * np.max(np.abs(uB))
    assert np.max(np.abs(uB[:, 0])) > 1e-9 * np.max(np.abs(uB))      # ... while at z = H the open top is not a wall
