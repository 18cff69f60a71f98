"""Pins for the oracle's partial-slip / moving-wall path (Appendix A; eqs 27, 46, 52; footnote 46).

* k = 0: closed forms — Couette flow between moving walls with slip, Poiseuille flow with slip under a uniform body force
  ((A12)), the bottom-wall plug flow of eq 52 with a moving wall;
* k != 0: the output satisfies the slip conditions (A1a), (A1b) u -/+ l du/dz = 0 on the walls, w = 0 there, continuity and the
  pressure-free curl of the momentum equation, checked with numpy's Chebyshev calculus on the oracle's output;
* limits: l -> 0 is the no-slip product; l -> infinity on the top wall (free slip) makes du/dz(H) vanish;
* the whole operator: a blob between moving walls is carried with the local Couette velocity; M stays symmetric with slip.
"""
from types import SimpleNamespace

import numpy as np
import numpy.polynomial.chebyshev as npcheb
import pytest

import oracle

BW, SC = 0, 1


def make_prob(wall_mode, H, nz, L=5.0, nxy=4, eta=1.3, **wall):
    return SimpleNamespace(wall_mode=wall_mode, Lx=L, Ly=L, H=H, nx=nxy, ny=nxy, nz=nz, w=6, beta_M=10.0, beta_D=12.0, eta=eta, **wall)


def wavenumbers(prob):
    kx = 2 * np.pi * np.arange(prob.nx // 2 + 1) / prob.Lx
    ny = prob.ny
    ky = 2 * np.pi * np.where(np.arange(ny) <= ny // 2, np.arange(ny), np.arange(ny) - ny) / prob.Ly
    return kx, ky


def test_couette_and_poiseuille_flow_with_slip_in_the_zero_mode():
    H, nz, eta = 3.0, 24, 1.7
    l0, lH, U0, UH = 0.4, 0.25, (0.3, -0.2), (1.1, 0.5)
    prob = make_prob(SC, H, nz, eta=eta, slip_0=l0, slip_H=lH, uwall_0=U0, uwall_H=UH)
    z = oracle.cheb_nodes(nz, H)
    nn = prob.nx * prob.ny
    # no force: u = a + b z with u(0) - l0 b = U0, u(H) + lH b = UH
    fh = np.zeros((3, nz, prob.ny, prob.nx // 2 + 1), dtype=complex)
    uh, _, _ = oracle.solve(prob, fh)
    for c in range(2):
        b = (UH[c] - U0[c]) / (H + l0 + lH)
        a = U0[c] + l0 * b
        assert np.max(np.abs(uh[c, :, 0, 0] / nn - (a + b * z))) < 1e-13
    assert np.max(np.abs(uh[2])) == 0.0 and np.max(np.abs(uh[:, :, 1:, :])) == 0.0      # a uniform wall velocity is a k = 0 datum
    # uniform body force G along x, walls at rest: u = -G z^2/(2 eta) + b z + a
    G = 0.9
    prob = make_prob(SC, H, nz, eta=eta, slip_0=l0, slip_H=lH)
    fh[0, :, 0, 0] = G * nn
    uh, _, _ = oracle.solve(prob, fh)
    # a - l0 b = 0 ; -G H^2/(2 eta) + b H + a + lH (-G H/eta + b) = 0
    b = (G * H * H / (2 * eta) + lH * G * H / eta) / (H + l0 + lH)
    a = l0 * b
    assert np.max(np.abs(uh[0, :, 0, 0] / nn - (-G * z * z / (2 * eta) + b * z + a))) < 1e-12
    # bottom wall moving, open top: plug flow (eq 52: du/dz(H) = 0)
    prob = make_prob(BW, H, nz, eta=eta, uwall_0=U0)
    uh, _, _ = oracle.solve(prob, np.zeros_like(fh))
    for c in range(2):
        assert np.max(np.abs(uh[c, :, 0, 0] / nn - U0[c])) < 1e-13


def _wall_source(prob, zs, seed=11):
    z = oracle.cheb_nodes(prob.nz, prob.H)
    shape = (3, prob.nz, prob.ny, prob.nx // 2 + 1)
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((3,) + shape[2:]) + 1j * rng.standard_normal((3,) + shape[2:])
    prof = z * np.exp(-(z / zs) ** 2) * (1 + 0.4 * z) + 0.7 * (prob.H - z) * np.exp(-((prob.H - z) / (0.8 * zs)) ** 2)
    return a[:, None, :, :] * prof[None, :, None, None]


@pytest.mark.parametrize("l0,lH", [(0.3, 0.0), (0.0, 0.5), (0.7, 0.2)])
def test_output_satisfies_the_slip_conditions_and_the_stokes_equations(l0, lH):
    H, nz = 6.0, 72
    prob = make_prob(SC, H, nz, L=6.0, slip_0=l0, slip_H=lH)
    fh = _wall_source(prob, 1.1)
    uh, wh, _ = oracle.solve(prob, fh, None, want_omega=True)
    z = oracle.cheb_nodes(nz, H)
    V = npcheb.chebvander(2 * z / H - 1, nz - 1)
    kxs, kys = wavenumbers(prob)

    def dz(nod, m=1):
        return npcheb.chebval(2 * z / H - 1, npcheb.chebder(np.linalg.solve(V, nod), m)) * (2 / H) ** m

    checked = 0
    for iy, ky in enumerate(kys):
        for ix, kx in enumerate(kxs):
            if (ix == 0 and iy == 0) or ix == prob.nx // 2 or iy == prob.ny // 2:
                continue
            k2 = kx * kx + ky * ky
            u, v, w = uh[0, :, iy, ix], uh[1, :, iy, ix], uh[2, :, iy, ix]
            scale = np.max(np.abs(uh[:, :, iy, ix]))
            for comp in (u, v):
                d = dz(comp)
                assert abs(comp[-1] - l0 * d[-1]) < 1e-9 * scale            # (A1a) at z = 0 (node l = nz-1)
                assert abs(comp[0] + lH * d[0]) < 1e-9 * scale              # (A1b) at z = H (node l = 0)
                if l0 > 0:
                    assert abs(comp[-1]) > 1e-4 * scale                     # the wall really slips
            assert abs(w[-1]) < 1e-11 * scale and abs(w[0]) < 1e-11 * scale
            f = fh[:, :, iy, ix]
            div = 1j * kx * u + 1j * ky * v + dz(w)
            assert np.max(np.abs(div)) < 1e-8 * np.max(np.abs(dz(w)))
            om2 = 2 * wh[:, :, iy, ix]
            curl_f = np.array([1j * ky * f[2] - dz(f[1]), dz(f[0]) - 1j * kx * f[2], 1j * kx * f[1] - 1j * ky * f[0]])
            for c in range(3):
                res = prob.eta * (dz(om2[c], 2) - k2 * om2[c]) + curl_f[c]
                assert np.max(np.abs(res)) < 1e-6 * np.max(np.abs(curl_f)), (ix, iy, c)
            checked += 1
    assert checked >= 3


def test_slip_length_limits():
    H, nz = 5.0, 64
    fh = _wall_source(make_prob(SC, H, nz, L=6.0), 1.0)
    ref, _, _ = oracle.solve(make_prob(SC, H, nz, L=6.0), fh)
    tiny, _, _ = oracle.solve(make_prob(SC, H, nz, L=6.0, slip_0=1e-9, slip_H=1e-9), fh)
    assert np.max(np.abs(tiny - ref)) < 1e-7 * np.max(np.abs(ref))            # l -> 0: no slip, continuously
    free, _, _ = oracle.solve(make_prob(SC, H, nz, L=6.0, slip_H=1e9), fh)    # l_H -> infinity: free-slip top wall
    z = oracle.cheb_nodes(nz, H)
    V = npcheb.chebvander(2 * z / H - 1, nz - 1)
    du = npcheb.chebval(1.0, npcheb.chebder(np.linalg.solve(V, free[0, :, 1, 1]))) * (2 / H)
    assert abs(du) < 1e-6 * np.max(np.abs(free[0, :, 1, 1])) and abs(free[0, 0, 1, 1]) > 1e-3 * np.max(np.abs(free[0, :, 1, 1]))


def test_a_blob_between_moving_walls_is_carried_by_the_couette_flow_and_slip_keeps_the_mobility_symmetric():
    h = 1.0
    wall = dict(slip_0=0.6, slip_H=0.3)
    base = dict(wall_mode=SC, Lx=24 * h, Ly=24 * h, H=10.0, nx=24, ny=24, nz=32, w=6, beta_M=6 * 1.327, beta_D=6 * 2.216, eta=1.0)
    pos = np.array([[5.2, 7.7, 4.1], [11.9, 12.3, 6.0]])
    # moving walls, no force: the blob velocity is the Couette profile averaged over its envelope = the profile at its centre
    # (a linear profile and an even, normalised envelope), up to the ES kernel's quadrature error
    U0, UH = (0.2, 0.0), (1.0, -0.4)
    prob = SimpleNamespace(**base, **wall, uwall_0=U0, uwall_H=UH)
    U, _ = oracle.mobility_apply(prob, pos, np.zeros((2, 3)), None, dft="fft")
    for c in range(2):
        b = (UH[c] - U0[c]) / (prob.H + wall["slip_0"] + wall["slip_H"])
        want = U0[c] + wall["slip_0"] * b + b * pos[:, 2]
        assert np.max(np.abs(U[:, c] - want)) < 2e-3 * max(abs(UH[c]), abs(U0[c]))
    assert np.max(np.abs(U[:, 2])) < 1e-12
    # with forces the product is affine: (M F + U_walls); M itself stays symmetric with slip
    prob0 = SimpleNamespace(**base, **wall)
    n = len(pos)
    M = np.zeros((3 * n, 3 * n))
    for j in range(n):
        for c in range(3):
            F = np.zeros((n, 3)); F[j, c] = 1.0
            M[:, 3 * j + c] = oracle.mobility_apply(prob0, pos, F, None, dft="fft")[0].ravel()
    assert np.linalg.norm(M - M.T) < 2e-4 * np.linalg.norm(M)
    assert np.linalg.eigvalsh(0.5 * (M + M.T)).min() > 0
    Mns = np.zeros_like(M)
    probn = SimpleNamespace(**base)
    for j in range(n):
        for c in range(3):
            F = np.zeros((n, 3)); F[j, c] = 1.0
            Mns[:, 3 * j + c] = oracle.mobility_apply(probn, pos, F, None, dft="fft")[0].ravel()
    assert np.all(np.diag(M)[[0, 1, 3, 4]] > np.diag(Mns)[[0, 1, 3, 4]])       # slipping walls resist tangential motion less
    F = np.random.default_rng(0).standard_normal((n, 3))
    Uaff, _ = oracle.mobility_apply(prob, pos, F, None, dft="fft")
    assert np.allclose(Uaff.ravel(), M @ F.ravel() + U.ravel(), rtol=0, atol=1e-12)
