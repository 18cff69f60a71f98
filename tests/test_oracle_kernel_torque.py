"""Pins for the oracle's kernel-derivative torque path (the paper's "second way"; footnotes 47-48).

Nothing in the paper prints a number for this path; what fixes it is
* the kernel derivative itself: phi' against difference quotients of the oracle's phi, the truncation point of footnote 47 as the
  minimum of |phi'| before the blow-up, found by brute-force scan;
* G = grad_x Delta_D^W against difference quotients of the oracle's own ``spread`` — with respect to the particle position in x, y
  (d/dx_p = -d/dx) and with respect to H in z (the Chebyshev nodes move as z_l = (H/2)(1 + xi_l), so d/dH samples the derivative
  with respect to the FIELD point, which is what decides the image sign of footnote 48);
* the cross product and the factor 1/2 of eq 7 / eq 11 by brute force over nodes, and exact weighted adjointness of the pair;
* the operator: M symmetric and positive definite by column assembly, mu^rt = mu^tr to five digits, every
  component -> 0 at the wall (footnote 48), and agreement with the Fourier-curl way to the method's 2-3 digits.
"""
import copy
import math
from types import SimpleNamespace

import numpy as np
import pytest

import oracle

BW, SC = 0, 1
BM, BD = 6 * 1.327, 6 * 2.216           # Table I, w = 6
RH_MD = 1.730


def box(wall_mode, nxy, nz, H, h=1.0, w=6, beta_M=BM, beta_D=BD, eta=1.0):
    return SimpleNamespace(wall_mode=wall_mode, Lx=nxy * h, Ly=nxy * h, H=H, nx=nxy, ny=nxy, nz=nz, w=w, beta_M=beta_M, beta_D=beta_D, eta=eta)


@pytest.mark.parametrize("beta", [BD, 4 * 1.785, 7.1])
def test_kernel_derivative_matches_difference_quotients_and_is_truncated_at_the_minimum(beta):
    alpha = 1.9
    ucut = oracle.es_dphi_cut(beta)
    assert 0.9 < ucut < 1.0
    s = np.linspace(-0.99 * ucut * alpha, 0.99 * ucut * alpha, 301)
    d = 1e-6
    fd = (oracle.es_phi(s + d, alpha, beta) - oracle.es_phi(s - d, alpha, beta)) / (2 * d)
    got = oracle.es_dphi(s, alpha, beta)
    assert np.max(np.abs(got - fd)) < 1e-8 * np.max(np.abs(fd))
    assert got[0] > 0 and got[-1] < 0 and abs(oracle.es_dphi(0.0, alpha, beta)) == 0.0     # odd, decreasing away from the centre
    # beyond the cut: zero (footnote 47), although phi itself is not
    out = np.array([ucut * alpha * (1 + 1e-12), 0.5 * (ucut + 1) * alpha, alpha])
    assert np.all(oracle.es_dphi(out, alpha, beta) == 0.0) and np.all(oracle.es_dphi(-out, alpha, beta) == 0.0)
    assert oracle.es_phi(out[1], alpha, beta) > 0
    # the cut is where |phi'| is smallest before it blows up: scan difference quotients of phi between the maximum of |phi'| and the edge
    u = np.linspace(0.9, 0.99999, 200001)
    dd = 1e-7
    mag = np.abs(oracle.es_phi(u * alpha + dd, alpha, beta) - oracle.es_phi(u * alpha - dd, alpha, beta)) / (2 * dd)
    imin = int(np.argmin(mag))
    assert 0 < imin < len(u) - 1
    assert abs(u[imin] - ucut) < 2e-4
    assert mag[-1] > 3 * mag[imin]                                                             # it does blow up beyond


def test_no_truncation_point_for_a_flat_kernel():
    assert math.isnan(oracle.es_dphi_cut(2.0))                                                 # |phi'| is monotone for beta <= 3 sqrt(3)/2


def _safe_particle(prob, rng, zlo, zhi):
    """a position none of whose nodes lies in the truncated shell or within 1e-3 h of the support edge (so that difference
    quotients of ``spread`` with respect to the particle position see a fixed set of nodes and the untruncated derivative)"""
    h = prob.Lx / prob.nx
    alpha = 0.5 * prob.w * h
    ucut = oracle.es_dphi_cut(prob.beta_D)
    zn = oracle.cheb_nodes(prob.nz, prob.H)
    while True:
        r = np.array([rng.uniform(0, prob.Lx), rng.uniform(0, prob.Ly), rng.uniform(zlo, zhi)])
        ok = True
        for c in (0, 1):
            d = np.abs(np.arange(-prob.nx, 2 * prob.nx) * h - r[c]) / alpha
            ok &= not np.any((d > ucut - 2e-3) & (d < 1 + 2e-3))
        for cz in (r[2], -r[2], 2 * prob.H - r[2]):
            d = np.abs(zn - cz) / alpha
            ok &= not np.any((d > ucut - 2e-3) & (d < 1 + 2e-3))
        if ok:
            return r


@pytest.mark.parametrize("wall_mode", [BW, SC])
def test_spread_curl_is_half_the_gradient_of_the_envelope_cross_the_torque(wall_mode):
    """(1/2) curl_x (tau Delta) = (1/2) grad Delta x tau (eq 7) with grad Delta from difference quotients of the oracle's own spread."""
    prob = box(wall_mode, 14, 15, 5.0, h=0.7, w=6, beta_D=9.3)
    rng = np.random.default_rng(5)
    h = prob.Lx / prob.nx
    for trial in range(3):
        r = _safe_particle(prob, rng, 0.3, 2.2 if wall_mode == BW else prob.H - 0.3)
        tau = rng.standard_normal(3)
        one = np.array([[1.0, 0.0, 0.0]])
        S = lambda pos, P=prob: oracle.spread(P, pos[None, :], one, P.beta_D)[0]
        d = 1e-6
        Gx = -(S(r + [d, 0, 0]) - S(r - [d, 0, 0])) / (2 * d)                  # d/dx = -d/dx_p
        Gy = -(S(r + [0, d, 0]) - S(r - [0, d, 0])) / (2 * d)
        # field-point z derivative: the nodes move with H, z_l = (H/2)(1 + xi_l); bottom wall only (in the slit H also moves the top image)
        if wall_mode == BW:
            Pp, Pm = copy.copy(prob), copy.copy(prob)
            dH = 1e-6
            Pp.H = prob.H + dH; Pm.H = prob.H - dH
            zn = oracle.cheb_nodes(prob.nz, prob.H)
            dS = (S(r, Pp) - S(r, Pm)) / (2 * dH)                              # = zeta'(z_l) z_l / H
            with np.errstate(divide="ignore", invalid="ignore"):
                Gz = np.where(zn[:, None, None] > 0, dS * prob.H / zn[:, None, None], 0.0)
        else:
            # slit: derivative with respect to the particle height flips the sign of the direct term only:
            # d/dz_p [phi(z - z_p) - phi(z + z_p) - phi(z - 2H + z_p)] = -phi'(z - z_p) - phi'(z + z_p) - phi'(z - 2H + z_p);
            # the field derivative is +phi'(z - z_p) - phi'(z + z_p) - phi'(z - 2H + z_p).  Take a particle whose images do not
            # reach the grid (both derivatives then differ by the sign only) — the image sign is pinned by the bottom-wall case.
            r = _safe_particle(prob, np.random.default_rng(100 + trial), 2.3, 2.7)
            Gx = -(S(r + [d, 0, 0]) - S(r - [d, 0, 0])) / (2 * d)
            Gy = -(S(r + [0, d, 0]) - S(r - [0, d, 0])) / (2 * d)
            Gz = -(S(r + [0, 0, d]) - S(r - [0, 0, d])) / (2 * d)
        G = np.stack([Gx, Gy, Gz])
        want = 0.5 * np.stack([G[1] * tau[2] - G[2] * tau[1], G[2] * tau[0] - G[0] * tau[2], G[0] * tau[1] - G[1] * tau[0]])
        got = oracle.spread_curl(prob, r[None, :], tau[None, :], prob.beta_D, np.zeros((3, prob.nz, prob.ny, prob.nx)))
        scale = np.max(np.abs(want))
        if wall_mode == BW:
            # the node on the wall (z_l = 0) does not move with H and cannot be sampled this way: compare the nodes above it
            assert np.max(np.abs(got[:, :-1] - want[:, :-1])) < 2e-7 * scale
        else:
            assert np.max(np.abs(got - want)) < 2e-7 * scale


def test_image_sign_of_the_z_derivative_makes_the_gradient_vanish_at_the_wall():
    """footnote 48: 'all components of the particle mobility go to zero at a wall': zeta'(l; z_p -> 0) -> 0."""
    prob = box(BW, 12, 17, 5.0, h=0.7)
    tau = np.array([[0.3, -1.1, 0.7]])
    z = np.zeros((3, prob.nz, prob.ny, prob.nx))
    g0 = oracle.spread_curl(prob, np.array([[3.3, 4.4, 0.0]]), tau, prob.beta_D, z.copy())
    assert np.all(g0 == 0.0)
    norms = [np.abs(oracle.spread_curl(prob, np.array([[3.3, 4.4, zp]]), tau, prob.beta_D, z.copy())).max() for zp in (1e-2, 1e-3, 1e-4)]
    assert norms[1] < 0.2 * norms[0] and norms[2] < 0.2 * norms[1]                 # linear in z_p
    u = np.random.default_rng(0).standard_normal(z.shape)
    assert np.all(oracle.interp_curl(prob, np.array([[3.3, 4.4, 0.0]]), u, prob.beta_D) == 0.0)
    probS = box(SC, 12, 17, 5.0, h=0.7)
    gH = oracle.spread_curl(probS, np.array([[3.3, 4.4, probS.H]]), tau, probS.beta_D, z.copy())
    assert np.max(np.abs(gH)) < 1e-15 * norms[0] / 1e-2


@pytest.mark.parametrize("wall_mode", [BW, SC])
def test_interp_curl_is_the_weighted_adjoint_of_spread_curl(wall_mode):
    prob = box(wall_mode, 14, 13, 4.0, h=0.7, w=4, beta_D=7.1)
    rng = np.random.default_rng(3)
    n = 17
    pos = np.stack([rng.uniform(-3, 20, n), rng.uniform(-3, 20, n), rng.uniform(0.0, prob.H, n)], axis=1)
    tau = rng.standard_normal((n, 3))
    u = rng.standard_normal((3, prob.nz, prob.ny, prob.nx))
    h = prob.Lx / prob.nx
    wq = (h * h * 0.5 * prob.H) * oracle.cc_weights(prob.nz)
    lhs = (oracle.interp_curl(prob, pos, u, prob.beta_D) * tau).sum()
    rhs = (u * oracle.spread_curl(prob, pos, tau, prob.beta_D, np.zeros_like(u)) * wq[None, :, None, None]).sum()
    assert lhs == pytest.approx(rhs, rel=1e-12)


def test_spread_curl_adds_to_the_force_field():
    prob = box(BW, 12, 11, 4.0, h=0.7, w=4, beta_D=7.1)
    pos = np.array([[1.1, 2.2, 1.3]])
    F, tau = np.array([[1.0, 2.0, 3.0]]), np.array([[0.5, -0.2, 0.1]])
    f = oracle.spread(prob, pos, F, prob.beta_M)
    t = oracle.spread_curl(prob, pos, tau, prob.beta_D, np.zeros_like(f))
    both = oracle.spread_curl(prob, pos, tau, prob.beta_D, f.copy())
    assert np.array_equal(both, f + t)


def _assemble(prob, pos, mode):
    n = len(pos)
    M = np.zeros((6 * n, 6 * n))
    for kind in (0, 1):
        for j in range(n):
            for c in range(3):
                F = np.zeros((n, 3)); T = np.zeros((n, 3))
                (F if kind == 0 else T)[j, c] = 1.0
                U, Om = oracle.mobility_apply(prob, pos, F, T, dft="fft", torque_mode=mode)
                M[: 3 * n, kind * 3 * n + 3 * j + c] = U.ravel()
                M[3 * n:, kind * 3 * n + 3 * j + c] = Om.ravel()
    return M


@pytest.mark.parametrize("wall_mode", [BW, SC])
def test_kernel_mode_mobility_is_symmetric_positive_definite_and_close_to_the_fourier_curl_way(wall_mode):
    h = 1.0 / 1.5
    prob = box(wall_mode, 30, 22, 9.0 if wall_mode == BW else 7.0, h)
    pos = np.array([[3.1, 4.2, 2.4], [6.0, 4.9, 3.3], [12.3, 15.0, 1.6]])       # non-overlapping, R_h = 1.15
    Mk = _assemble(prob, pos, "kernel")
    asym = np.linalg.norm(Mk - Mk.T) / np.linalg.norm(Mk)
    assert asym < 2e-4
    ev = np.linalg.eigvalsh(0.5 * (Mk + Mk.T))
    assert ev.min() > 1e-3 * ev.max() > 0                                       # SPD
    n3 = 3 * len(pos)
    assert np.array_equal(Mk[:n3, :n3], _assemble_tt(prob, pos))                # forces -> velocities do not depend on the torque path
    Mf = _assemble(prob, pos, "fourier")
    # "both preserve the desired accuracy": 2-3 digits, block by block in the blocks' own scale
    for (a, b) in ((slice(0, n3), slice(n3, None)), (slice(n3, None), slice(0, n3)), (slice(n3, None), slice(n3, None))):
        assert np.max(np.abs(Mk[a, b] - Mf[a, b])) < 2e-2 * np.max(np.abs(Mf[a, b]))


def _assemble_tt(prob, pos):
    n = len(pos)
    M = np.zeros((3 * n, 3 * n))
    for j in range(n):
        for c in range(3):
            F = np.zeros((n, 3)); F[j, c] = 1.0
            U, _ = oracle.mobility_apply(prob, pos, F, np.zeros((n, 3)), dft="fft", torque_mode="kernel")
            M[:, 3 * j + c] = U.ravel()
    return M


def test_kernel_mode_tr_and_rt_self_couplings_agree_to_five_digits_and_rr_matches_the_sphere():
    """PAPER.md:450 ('well within five digits', in units of 1/(6 pi eta R_h^2)) holds for the kernel-derivative way as well: spreading
    and interpolation are exact adjoints; 8 pi eta R_h^3 mu^rr -> 1 away from walls with the same dipole R_h."""
    h = 1.0
    Rh = RH_MD * h
    prob = box(BW, 132, 54, 19.2 * Rh, h)
    norm = 6 * math.pi * prob.eta * Rh ** 2
    pos = np.array([[30.3, 40.1, 1.5 * Rh]])
    U, _ = oracle.mobility_apply(prob, pos, np.zeros((1, 3)), np.array([[1.0, 0, 0]]), dft="fft", torque_mode="kernel")
    _, Om = oracle.mobility_apply(prob, pos, np.array([[0, 1.0, 0]]), np.zeros((1, 3)), dft="fft", torque_mode="kernel")
    assert abs(U[0, 1] - Om[0, 0]) * norm < 1e-5
    assert abs(U[0, 1]) * norm > 1e-3 and U[0, 1] < 0
    Uf, _ = oracle.mobility_apply(prob, pos, np.zeros((1, 3)), np.array([[1.0, 0, 0]]), dft="fft", torque_mode="fourier")
    assert U[0, 1] == pytest.approx(Uf[0, 1], rel=2e-2)
    far = np.array([[30.3, 40.1, 9.0 * Rh]])
    _, Omr = oracle.mobility_apply(prob, far, np.zeros((1, 3)), np.array([[0, 0, 1.0]]), dft="fft", torque_mode="kernel")
    assert Omr[0, 2] * 8 * math.pi * prob.eta * Rh ** 3 == pytest.approx(1.0, rel=2e-2)
