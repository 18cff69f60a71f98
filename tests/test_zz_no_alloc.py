"""dp_bin_particles_static — the product's particle sort for callers that are not allowed to allocate device memory.

Who needs it: code that runs inside an application which handed all of HBM to its own memory pool at start-up (a later cudaMalloc
fails or fragments that pool), plug-ins and latency-bound loops whose host forbids driver allocations after initialisation
(cudaMalloc / cudaFree may synchronise the whole device), workers that only ever receive buffers.  A plan gets the work arrays of its
counting sort from cudaMalloc in dp_create; this entry point keeps them in a fixed 2.5 MiB array that is part of libdpstokes.so, so it
needs no plan and allocates nothing — at the price of a size limit (262,144 particles, 131,072 tiles) and of one array shared by
every call on a device (calls that overlap on the GPU race; the array keeps the previous call's contents).

The test compares it with the sort the product itself performs (read back through dp_copy_bins_to_host) on the same positions.
Integer work: tile_start must be bit-identical; perm must hold the same particles in every tile (the order inside one tile comes
from atomic counters on both sides and is not defined).  Two calls in a row with DIFFERENT inputs — the second smaller — show that
what the first call left in the shared array does not leak into the second.

This file sorts last on purpose (pytest -x stops at the first failure; a failure here hides nothing behind it)."""
import dataclasses

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dp():
    import torch
    assert torch.cuda.is_available()
    import paper_2210_01837_b200 as dp
    dp.load_library()          # fails loudly if the extension is missing
    return dp


def canonical(perm, start):
    """Particles of every tile in ascending index order: the part of (perm, tile_start) that is uniquely defined."""
    perm = np.asarray(perm, dtype=np.int64)
    start = np.asarray(start, dtype=np.int64)
    tile_of_slot = np.repeat(np.arange(len(start) - 1), np.diff(start))
    return perm[np.lexsort((perm, tile_of_slot))]


def product_sort(dp, prob, pos):
    """The existing path: one product's binning stage (dp_debug_run_stage up to spreading), sort read back from the plan."""
    import torch
    n = len(pos)
    F = np.ones((n, 3))
    with dp.Plan(prob, max_particles=n, use_torques=False) as plan:
        dpos, dF = torch.from_numpy(pos).cuda(), torch.from_numpy(F).cuda()
        plan.run_stage(dpos, dF, None, 1)
        torch.cuda.synchronize()
        return plan.copy_bins(n), plan.params


def test_static_binning_matches_the_products_sort_on_two_calls_in_a_row(dp):
    import torch
    # call 1: slit, 4000 particles on a 192 x 192 grid (12 x 48 tiles); some x, y outside [0, L) (wrapped) and three particles out of the domain
    prob1, pos1, _, _ = workloads.random_slit(n=4000, L=128.0, nxy=192, nz=48, H=8.0, seed=5, name="noalloc-1")
    pos1 = np.ascontiguousarray(pos1)
    pos1[::7, 0] += 3 * 128.0
    pos1[::11, 1] -= 2 * 128.0
    pos1[[5, 900, 3999], 2] = [-0.5, 9.0, 8.5]
    # call 2: bottom wall, fewer particles, ragged grid (60 x 60: 4 x 15 tiles, the last tile column 12 nodes wide), all in one corner
    prob2, pos2, _, _ = workloads.config(1)
    prob2 = dataclasses.replace(prob2, nx=60, ny=60, Lx=40.0, Ly=40.0, has_torque=False)
    rng = np.random.default_rng(12)
    pos2 = np.column_stack([rng.uniform(0, 9.0, 777), rng.uniform(31.0, 40.0, 777), rng.uniform(0.5, 3.0, 777)])

    (perm_ref1, start_ref1), params1 = product_sort(dp, prob1, pos1)
    (perm_ref2, start_ref2), params2 = product_sort(dp, prob2, pos2)
    assert start_ref1[-1] == len(pos1) and start_ref2[-1] == len(pos2)

    # the two calls, back to back on one stream, outputs read only after both were issued
    d1, d2 = torch.from_numpy(pos1).cuda(), torch.from_numpy(pos2).cuda()
    perm1, start1 = dp.bin_particles_static(params1, d1)
    perm2, start2 = dp.bin_particles_static(params2, d2)
    torch.cuda.synchronize()
    for (perm, start), (perm_ref, start_ref) in (((perm1, start1), (perm_ref1, start_ref1)), ((perm2, start2), (perm_ref2, start_ref2))):
        perm, start = perm.cpu().numpy(), start.cpu().numpy()
        assert np.array_equal(start, start_ref)                                   # bit-exact
        assert np.array_equal(np.sort(perm), np.arange(len(perm)))                # a permutation
        assert np.array_equal(canonical(perm, start), canonical(perm_ref, start_ref))

    # and once more with the first input: the array now holds call 2's leftovers
    perm3, start3 = dp.bin_particles_static(params1, d1)
    torch.cuda.synchronize()
    assert np.array_equal(start3.cpu().numpy(), start_ref1)
    assert np.array_equal(canonical(perm3.cpu().numpy(), start_ref1), canonical(perm_ref1, start_ref1))


def test_static_binning_rejects_what_does_not_fit_its_fixed_array(dp):
    """Sizes beyond the fixed array are refused with their own error code before anything is launched (the pointers are never touched)."""
    import ctypes
    import torch
    L = dp.load_library()
    prob, pos, _, _ = workloads.config(1)
    with dp.Plan(prob, max_particles=8, use_torques=False) as plan:
        params = plan.params
    out = torch.zeros(4, dtype=torch.int32, device="cuda")
    vp = lambda t: ctypes.c_void_p(t.data_ptr())
    too_many = dp.binding.STATIC_BIN_MAX_PARTICLES + 1
    assert L.dp_bin_particles_static(ctypes.byref(params), too_many, vp(out), vp(out), vp(out), None) == dp.binding.ETOOBIG
    big = dp.binding.dp_params.from_buffer_copy(params)
    big.nx = big.ny = 4320                    # config 5's grid: 270 x 1080 = 291,600 tiles
    big.Lx = big.Ly = 4320 * (params.Lx / params.nx)
    assert L.dp_bin_particles_static(ctypes.byref(big), 4, vp(out), vp(out), vp(out), None) == dp.binding.ETOOBIG
    assert b"fixed work array" in L.dp_strerror(dp.binding.ETOOBIG)
    assert L.dp_bin_particles_static(ctypes.byref(params), -1, vp(out), vp(out), vp(out), None) == -1
    torch.cuda.synchronize()
    assert int(out.sum()) == 0
