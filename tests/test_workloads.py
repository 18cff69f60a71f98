"""Seeded input recipes (workloads/): the non-overlapping jittered-lattice stand-in of SURVEY.md §8(d) and the stability of BASELINE.json's own draws."""
import hashlib

import numpy as np
import pytest

import workloads


def min_inplane_distance(pos, L):
    from scipy.spatial import cKDTree
    xy = np.mod(pos[:, :2], L)
    d, _ = cKDTree(xy, boxsize=L).query(xy, k=2)
    return float(d[:, 1].min())


def test_jittered_lattice_has_no_overlaps_and_keeps_the_recipe():
    n = 16384
    prob_u, pos_u, F_u, T_u = workloads.monolayer_bw(n=n, seed=7)
    prob_j, pos_j, F_j, T_j = workloads.monolayer_bw(n=n, seed=7, xy="jittered")
    assert prob_j == prob_u                                            # same box, grid, kernels
    assert np.array_equal(pos_j[:, 2], pos_u[:, 2]) and np.array_equal(F_j, F_u) and np.array_equal(T_j, T_u)   # same heights and drives
    L = prob_j.Lx
    assert pos_j.shape == (n, 3) and pos_j[:, :2].min() >= 0.0 and pos_j[:, :2].max() < L
    assert min_inplane_distance(pos_j, L) >= 2.0 * prob_j.a           # hard-disk constraint (periodic images included)
    assert min_inplane_distance(pos_u, L) < 0.5                        # the uniform draw overlaps: that is what the stand-in removes
    assert abs(n * np.pi / L ** 2 - 0.4) < 1e-12                       # area fraction 0.4
    again = workloads.monolayer_bw(n=n, seed=7, xy="jittered")[1]
    assert np.array_equal(again, pos_j)                                # seeded
    # index order carries no spatial order (shuffled sites): neighbours in index are far apart on average
    assert np.median(np.abs(np.diff(pos_j[:, 0]))) > 0.1 * L


def test_jittered_lattice_rejects_what_it_cannot_place():
    with pytest.raises(ValueError):
        workloads.monolayer_bw(n=1000, xy="jittered")                  # not a square number
    with pytest.raises(ValueError):
        workloads.monolayer_bw(n=1024, xy="poisson")


def test_config_draws_are_stable():
    """BASELINE.json's configs are what every stored comparison refers to: adding recipes must not move them."""
    prob, pos, F, T = workloads.config(3)
    assert (prob.nx, prob.ny, prob.nz, len(pos)) == (1080, 1080, 32, 65536)
    assert hashlib.md5(pos.tobytes()).hexdigest() == hashlib.md5(workloads.monolayer_bw()[1].tobytes()).hexdigest()
    p1, pos1, F1, _ = workloads.config(1)
    assert pos1.shape == (128, 3) and 1.5 <= pos1[:, 2].min() and pos1[:, 2].max() <= 5.0
