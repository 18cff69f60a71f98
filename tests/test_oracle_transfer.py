"""Pins for the oracle's particle <-> grid transfer (O1 spread, O12 interpolate; eqs 7, 9, 10).

Checked against: a brute-force evaluation of Delta^W at EVERY grid node and every periodic image (no support / wrap
logic), exact structural invariants (adjointness, wall nulling, grid-cell translation, slit mirror symmetry), and
the continuum facts int Delta = 1 and int z Delta = z_p.
"""
from types import SimpleNamespace

import numpy as np
import pytest

import oracle

BW, SC = 0, 1


def prob_small(wall_mode, nx=12, ny=10, nz=11, h=0.7, H=4.0, w=4, beta=7.1):
    return SimpleNamespace(wall_mode=wall_mode, Lx=nx * h, Ly=ny * h, H=H, nx=nx, ny=ny, nz=nz, w=w, beta_M=beta, beta_D=beta * 1.3, eta=1.0)


@pytest.mark.parametrize("wall_mode", [BW, SC])
def test_spread_equals_brute_force_over_all_nodes_and_images(wall_mode):
    prob = prob_small(wall_mode)
    h, alpha = prob.Lx / prob.nx, 0.5 * prob.w * prob.Lx / prob.nx
    pos = np.array([[0.13, 0.2, 0.9],                       # footprint wraps below 0 in x and y, overlaps the wall
                    [prob.Lx - 0.05, 3.3, 2.0],             # wraps above Lx
                    [4.0 + 17 * prob.Lx, -2 * prob.Ly + 1.234, prob.H - 0.6],   # far outside the primary cell; near the top
                    [2.8, 2.1, 0.0]])                       # ON the wall: contributes nothing
    val = np.array([[1.0, -2.0, 0.5], [0.3, 0.7, -1.1], [2.0, 0.1, 0.4], [5.0, 5.0, 5.0]])
    got = oracle.spread(prob, pos, val, prob.beta_M)
    z = oracle.cheb_nodes(prob.nz, prob.H)
    xg = np.arange(prob.nx) * h
    yg = np.arange(prob.ny) * h
    want = np.zeros_like(got)
    phi = lambda s: oracle.es_phi(np.ravel(s), alpha, prob.beta_M).reshape(np.shape(s))
    for p in range(len(pos)):
        px = sum(phi(xg - pos[p, 0] + m * prob.Lx) for m in range(-30, 31))     # periodic sum, all images
        py = sum(phi(yg - pos[p, 1] + m * prob.Ly) for m in range(-30, 31))
        zeta = phi(z - pos[p, 2]) - phi(z + pos[p, 2])                            # eq 9: minus the image in z = 0
        if wall_mode == SC:
            zeta = zeta - phi(z - (2 * prob.H - pos[p, 2]))                        # and in z = H
        want += val[p][:, None, None, None] * zeta[None, :, None, None] * py[None, None, :, None] * px[None, None, None, :]
    assert np.max(np.abs(got - want)) < 1e-14 * np.max(np.abs(want))
    assert np.count_nonzero(got[0, :, 0, 0]) < prob.nz      # compact in z as well


@pytest.mark.parametrize("wall_mode", [BW, SC])
def test_interp_is_the_weighted_adjoint_of_spread(wall_mode):
    """<interp(u), F> = sum_g u(g) spread(F)(g) h^2 (H/2) w_l  exactly (P5 iv; PAPER.md:333 'the same grid values')."""
    prob = prob_small(wall_mode, nx=14, ny=14, nz=13)
    rng = np.random.default_rng(0)
    n = 17
    pos = np.stack([rng.uniform(-3, 20, n), rng.uniform(-3, 20, n), rng.uniform(0.0, prob.H, n)], axis=1)
    F = rng.standard_normal((n, 3))
    u = rng.standard_normal((3, prob.nz, prob.ny, prob.nx))
    h = prob.Lx / prob.nx
    wq = (h * h * 0.5 * prob.H) * oracle.cc_weights(prob.nz)
    lhs = (oracle.interp(prob, pos, u, prob.beta_D) * F).sum()
    rhs = (u * oracle.spread(prob, pos, F, prob.beta_D) * wq[None, :, None, None]).sum()
    assert lhs == pytest.approx(rhs, rel=1e-13)


def test_particle_on_the_wall_spreads_and_feels_nothing():
    """z_p = 0: Delta^W = 0 identically (eq 9), for both envelopes."""
    prob = prob_small(BW)
    pos = np.array([[1.0, 2.0, 0.0]])
    assert np.all(oracle.spread(prob, pos, np.ones((1, 3)), prob.beta_M) == 0.0)
    u = np.random.default_rng(1).standard_normal((3, prob.nz, prob.ny, prob.nx))
    assert np.all(oracle.interp(prob, pos, u, prob.beta_M) == 0.0)
    probS = prob_small(SC)
    posH = np.array([[1.0, 2.0, probS.H]])
    assert np.max(np.abs(oracle.spread(probS, posH, np.ones((1, 3)), probS.beta_M))) < 1e-16


def test_translation_by_one_cell_rolls_the_grid():
    prob = prob_small(BW)
    h = prob.Lx / prob.nx
    rng = np.random.default_rng(2)
    pos = np.stack([rng.uniform(0, prob.Lx, 9), rng.uniform(0, prob.Ly, 9), rng.uniform(0.2, 3.0, 9)], axis=1)
    F = rng.standard_normal((9, 3))
    g0 = oracle.spread(prob, pos, F, prob.beta_M)
    g1 = oracle.spread(prob, pos + np.array([2 * h, -3 * h, 0.0]), F, prob.beta_M)
    assert np.max(np.abs(np.roll(g0, (-3, 2), axis=(2, 3)) - g1)) < 1e-12 * np.max(np.abs(g0))


def test_slit_mirror_symmetry_of_the_spread_field():
    """The Chebyshev grid is symmetric under z -> H - z (l -> nz-1-l); so is the doubly-imaged envelope."""
    prob = prob_small(SC, nz=12)
    rng = np.random.default_rng(3)
    pos = np.stack([rng.uniform(0, prob.Lx, 7), rng.uniform(0, prob.Ly, 7), rng.uniform(0.1, prob.H - 0.1, 7)], axis=1)
    F = rng.standard_normal((7, 3))
    g0 = oracle.spread(prob, pos, F, prob.beta_M)
    posm = pos.copy()
    posm[:, 2] = prob.H - pos[:, 2]
    g1 = oracle.spread(prob, posm, F, prob.beta_M)
    assert np.max(np.abs(g0[:, ::-1] - g1)) < 1e-12 * np.max(np.abs(g0))


def test_moments_of_the_spread_field():
    """Away from walls int Delta dx = 1 and int z Delta dx = z_p (eq 53-54: unit mass, symmetric), evaluated with the
    method's own quadrature (trapezoid x Clenshaw-Curtis) to the paper's 2-3 digits."""
    nx = ny = 24
    nz = 32
    h = 1.0 / 1.5
    prob = SimpleNamespace(wall_mode=BW, Lx=nx * h, Ly=ny * h, H=13.0, nx=nx, ny=ny, nz=nz, w=6, beta_M=6 * 1.714, beta_D=6 * 2.216, eta=1.0)
    zq = (h * h * 0.5 * prob.H) * oracle.cc_weights(nz)
    z = oracle.cheb_nodes(nz, prob.H)
    for zp in (3.1, 5.0, 6.6):
        pos = np.array([[3.37, 8.11, zp]])
        g = oracle.spread(prob, pos, np.array([[1.0, 2.0, -3.0]]), prob.beta_M)
        tot = (g * zq[None, :, None, None]).sum(axis=(1, 2, 3))
        assert np.allclose(tot, [1.0, 2.0, -3.0], rtol=5e-3)
        zbar = (g[0] * (zq * z)[:, None, None]).sum()
        assert zbar == pytest.approx(zp, rel=5e-3)
