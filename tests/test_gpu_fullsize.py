"""Full-size GPU parity: BASELINE.json configs 3, 4 and 5 exactly as ``workloads.config(i)`` produces them (the launch
configuration bench.py times), through the C ABI, against the CPU oracle.

* configs 3 and 4: the whole oracle product (``oracle.mobility_apply``, xy transforms by the oracle's own plain FFT, which is
  pinned against its naive sums in tests/test_oracle_basics.py); bar: stacked (U, Omega) relative L2 <= 1e-10 (north_star) AND
  a per-particle bound max|dU| <= 1e-9 max|U| (one wrong particle in a million is invisible in an L2 norm).
* config 5 (N = 1,048,576, 4320 x 4320 x 32): stage by stage at full size, every stage fed with the CUDA path's previous
  stage: oracle spread of ALL particles vs the CUDA grids, plane by plane; sampled planes of the forward and inverse xy
  transforms vs the oracle's FFT; the per-wavenumber solve on sampled (kx, ky) columns (lowest modes, k = 0, both Nyquist
  lines, random interior) vs ``oracle.solve_modes``; oracle interpolation of the CUDA path's real-space u, omega for ALL particles
  vs the CUDA U, Omega.  The whole oracle product at config 5 (about 60 GB of host memory, two minutes) runs too, unless
  DP_FULL_ORACLE_CFG5=0.
* the fp32 spread / interpolate variant (transfer_fp32 = 1, north_star: <= 1e-5) at configs 3, 4 and 5 in the torque mode bench.py times,
  against the same whole-oracle results.
"""
import os
import sys

import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-10          # north_star: relative L2 of the stacked output, fp64
TOL_MAX = 1e-9       # per-particle: max |difference| / max |reference|


def rel_l2(a, b):
    a = np.asarray(a); b = np.asarray(b)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def rel_max(a, b):
    return float(np.abs(np.asarray(a) - np.asarray(b)).max() / np.abs(np.asarray(b)).max())


@pytest.fixture(scope="module")
def dp():
    import torch
    assert torch.cuda.is_available()
    import paper_2210_01837_b200 as dp
    dp.load_library()
    return dp


def to_dev(*arrs):
    import torch
    return [None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]


def check_product(U, Om, U_o, Om_o):
    stacked = rel_l2(np.concatenate([U, Om], axis=1), np.concatenate([U_o, Om_o], axis=1))
    assert stacked < TOL, stacked
    assert rel_l2(U, U_o) < TOL and rel_l2(Om, Om_o) < TOL
    assert rel_max(U, U_o) < TOL_MAX and rel_max(Om, Om_o) < TOL_MAX, (rel_max(U, U_o), rel_max(Om, Om_o))
    return stacked


TOL_FP32 = 1e-5      # north_star: the optional fp32 spread / interpolate variant, relative L2
TOL_FP32_MAX = 1e-4  # per particle, of max |reference| (fp32 rounding, 6e-8, of ~10^3 accumulated terms each way; measured: see the printed line)


def run_fp32_variant(dp, prob, pos, F, T, torque_mode):
    """The same product on a transfer_fp32 plan (fp32 spreading, interpolation and real-space grids; transforms and solves fp64)."""
    import torch
    with dp.Plan(prob, max_particles=len(pos), use_torques=True, torque_mode=1 if torque_mode == "kernel" else 0, transfer_fp32=True) as plan:
        U, Om = plan.mobility_apply(*to_dev(pos, F, T))
        torch.cuda.synchronize()
        assert plan.check() == 0
        U, Om = U.cpu().numpy(), Om.cpu().numpy()
    torch.cuda.empty_cache()
    return U, Om


def check_fp32_product(tag, U, Om, U_o, Om_o):
    stacked = rel_l2(np.concatenate([U, Om], axis=1), np.concatenate([U_o, Om_o], axis=1))
    print("%s fp32 transfer variant: stacked rel L2 %.2e, per-particle max %.2e / %.2e" % (tag, stacked, rel_max(U, U_o), rel_max(Om, Om_o)))
    assert stacked < TOL_FP32, stacked
    assert rel_l2(U, U_o) < TOL_FP32 and rel_l2(Om, Om_o) < TOL_FP32
    assert rel_max(U, U_o) < TOL_FP32_MAX and rel_max(Om, Om_o) < TOL_FP32_MAX, (rel_max(U, U_o), rel_max(Om, Om_o))


@pytest.mark.parametrize("cfg,torque_mode", [(3, "fourier"), (4, "fourier"), (3, "kernel"), (4, "kernel")])
def test_cfg3_cfg4_full_size_against_the_oracle(dp, cfg, torque_mode):
    """torque_mode: "fourier" = curl in Fourier-Chebyshev space (6 fields), "kernel" = ES kernel derivative (3 fields, bench.py's default)"""
    import torch
    prob, pos, F, T = workloads.config(cfg)
    assert len(pos) == {3: 65536, 4: 262144}[cfg] and prob.nx == {3: 1080, 4: 2160}[cfg] and prob.nz == {3: 32, 4: 48}[cfg]
    with dp.Plan(prob, max_particles=len(pos), use_torques=True, torque_mode=1 if torque_mode == "kernel" else 0) as plan:
        assert plan.fft_backend() == "own"
        U, Om = plan.mobility_apply(*to_dev(pos, F, T))
        torch.cuda.synchronize()
        assert plan.check() == 0
        U, Om = U.cpu().numpy(), Om.cpu().numpy()
    torch.cuda.empty_cache()
    fp32 = run_fp32_variant(dp, prob, pos, F, T, torque_mode) if torque_mode == "kernel" else None   # the variant bench.py times, same oracle run
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft", torque_mode=torque_mode)
    if fp32 is not None:
        check_fp32_product("cfg%d (%s)" % (cfg, torque_mode), fp32[0], fp32[1], U_o, Om_o)
    err = check_product(U, Om, U_o, Om_o)
    print("cfg%d (%s) full size: stacked rel L2 %.2e, per-particle max %.2e / %.2e" % (cfg, torque_mode, err, rel_max(U, U_o), rel_max(Om, Om_o)))


def _sample_modes(prob, rng, n_random=3000):
    nx, ny = prob.nx, prob.ny
    nkx = nx // 2 + 1
    modes = set()
    for ix in range(0, 4):                               # lowest modes incl. k = 0 and negative ky
        for iy in list(range(0, 4)) + [ny - 1, ny - 2, ny - 3]:
            modes.add((ix, iy))
    for iy in rng.integers(0, ny, 40):                   # the kx Nyquist line and kx = 0 line
        modes.add((nx // 2, int(iy)))
        modes.add((0, int(iy)))
    for ix in rng.integers(0, nkx, 40):                  # the ky Nyquist line
        modes.add((int(ix), ny // 2))
    modes.add((nx // 2, ny // 2))
    modes.add((nx // 2, 0))
    modes.add((0, ny // 2))
    for ix, iy in zip(rng.integers(0, nkx, n_random), rng.integers(0, ny, n_random)):
        modes.add((int(ix), int(iy)))
    m = np.array(sorted(modes), dtype=np.int32)
    return m[:, 0].copy(), m[:, 1].copy()


def test_cfg5_full_size_stage_by_stage_against_the_oracle(dp):
    import torch
    prob, pos, F, T = workloads.config(5)
    n = len(pos)
    assert n == 1048576 and (prob.nx, prob.ny, prob.nz) == (4320, 4320, 32)
    nz, ny, nx = prob.nz, prob.ny, prob.nx
    dpos, dF, dT = to_dev(pos, F, T)
    rng = np.random.default_rng(55)
    with dp.Plan(prob, max_particles=n, use_torques=True) as plan:
        assert plan.fft_backend() == "own"
        # ---- step 1: oracle spread of all 1,048,576 particles vs the CUDA grids, plane by plane
        plan.run_stage(dpos, dF, dT, 1)
        sample_planes = [(0, nz - 2), (2, nz - 5), (4, nz - 3), (1, nz - 9)]        # (field, l): near the wall, where the monolayer sits (t_x = t_z = 0 here: torques are +y)
        kept = {}
        for grp, (val, beta) in enumerate(((F, prob.beta_M), (T, prob.beta_D))):
            ref = oracle.spread(prob, pos, val, beta)                               # [3, nz, ny, nx]
            num = den = 0.0
            worst = 0.0
            for c in range(3):
                for l in range(nz):
                    g = plan.copy_plane(0, 3 * grp + c, l)
                    d = g - ref[c, l]
                    num += float((d * d).sum()); den += float((ref[c, l] ** 2).sum())
                    worst = max(worst, float(np.abs(d).max()))
                    if (3 * grp + c, l) in sample_planes:
                        kept[(3 * grp + c, l)] = g.copy()
            # the two sides differ in summation order and in the rounding of the ES exponent beta (sqrt(1 - q^2) - 1): one ulp in q
            # (s * (1/alpha) here, s / alpha in the oracle; fused 1 - q q) is amplified by beta / (2 sqrt(1 - q^2)) <~ 100
            assert np.sqrt(num / den) < 5e-13 and worst < 2e-12 * float(np.abs(ref).max()), (grp, np.sqrt(num / den), worst)
            del ref
        # ---- step 2 (xy): sampled planes of the forward spectrum vs the oracle's FFT of the (verified) grid planes;
        #      the nodal columns of the sampled modes are gathered from all planes for the solve check
        plan.run_stage(dpos, dF, dT, 2)
        keys = sorted(kept)
        ref = oracle.dft_xy_forward(np.stack([kept[k] for k in keys]), "fft")      # one call: the planes run in parallel threads
        for i, (f, l) in enumerate(keys):
            spec = plan.copy_plane(1, f, l)
            assert rel_l2(spec, ref[i]) < 1e-13, (f, l, rel_l2(spec, ref[i]))
        del ref, kept
        ix, iy = _sample_modes(prob, rng)
        cols = np.empty((6, nz, len(ix)), dtype=np.complex128)
        for f in range(6):
            for l in range(nz):
                cols[f, l] = plan.copy_plane(1, f, l)[iy, ix]
        # ---- steps 2(z)-6: the solve on the sampled columns (the kernel folds 1/(nx ny) into its output)
        uh_o, wh_o = oracle.solve_modes(prob, ix, iy, cols[:3], cols[3:], want_omega=True)
        plan.run_stage(dpos, dF, dT, 3)
        out = np.empty((6, nz, len(ix)), dtype=np.complex128)
        inv_planes = {}
        for f in range(6):
            for l in range(nz):
                pl = plan.copy_plane(1, f, l)
                out[f, l] = pl[iy, ix]
                if (f, l) in sample_planes:
                    inv_planes[(f, l)] = pl.copy()
        out *= nx * ny
        ref = np.concatenate([uh_o, wh_o])
        assert rel_l2(out, ref) < 1e-11, rel_l2(out, ref)
        col_err = np.sqrt((np.abs(out - ref) ** 2).sum(axis=(0, 1)) / (np.abs(ref) ** 2).sum(axis=(0, 1)).clip(1e-300))
        col_scale = np.sqrt((np.abs(ref) ** 2).sum(axis=(0, 1)))
        big = col_scale > 1e-6 * col_scale.max()                                     # columns that carry signal
        assert col_err[big].max() < 1e-9, float(col_err[big].max())                 # every sampled column on its own
        k0 = np.where((ix == 0) & (iy == 0))[0]
        assert len(k0) == 1 and col_err[k0[0]] < 1e-11
        # ---- step 7: sampled planes of the real-space result vs the oracle's inverse FFT of the CUDA solve output
        plan.run_stage(dpos, dF, dT, 4)
        keys = sorted(inv_planes)
        back = oracle.dft_xy_inverse(np.stack([inv_planes[k] for k in keys]), nx, "fft") * (nx * ny)   # the oracle's inverse carries 1/(nx ny); the kernel already applied it
        for i, (f, l) in enumerate(keys):
            g = plan.copy_plane(0, f, l)
            assert rel_l2(g, back[i]) < 1e-13, (f, l, rel_l2(g, back[i]))
        del back, inv_planes
        # ---- step 8: oracle interpolation of the CUDA path's real-space u, omega for ALL particles vs the CUDA U, Omega
        grid = np.empty((6, nz, ny, nx))
        for f in range(6):
            for l in range(nz):
                grid[f, l] = plan.copy_plane(0, f, l)
        U, Om = plan.mobility_apply(dpos, dF, dT)
        torch.cuda.synchronize()
        assert plan.check() == 0
        U, Om = U.cpu().numpy(), Om.cpu().numpy()
        U_o = oracle.interp(prob, pos, grid[:3], prob.beta_M)
        Om_o = oracle.interp(prob, pos, grid[3:], prob.beta_D)
        del grid
        assert rel_l2(U, U_o) < 1e-12 and rel_l2(Om, Om_o) < 1e-12, (rel_l2(U, U_o), rel_l2(Om, Om_o))
        assert rel_max(U, U_o) < 1e-11 and rel_max(Om, Om_o) < 1e-11


@pytest.mark.skipif(os.environ.get("DP_FULL_ORACLE_CFG5") == "0", reason="whole oracle product at config 5 switched off (DP_FULL_ORACLE_CFG5=0)")
@pytest.mark.parametrize("torque_mode", ["kernel", "fourier"])
def test_cfg5_whole_product_against_the_whole_oracle(dp, torque_mode):
    """Config 5 as bench.py runs it (default torque mode "kernel"; "fourier" is its second timed form) against the WHOLE oracle
    product (up to about 60 GB of host memory and two minutes on the 16-core GPU box; DP_FULL_ORACLE_CFG5=0 skips it on a smaller host)."""
    import torch
    prob, pos, F, T = workloads.config(5)
    with dp.Plan(prob, max_particles=len(pos), use_torques=True, torque_mode=1 if torque_mode == "kernel" else 0) as plan:
        U, Om = plan.mobility_apply(*to_dev(pos, F, T))
        torch.cuda.synchronize()
        assert plan.check() == 0
        U, Om = U.cpu().numpy(), Om.cpu().numpy()
    torch.cuda.empty_cache()
    fp32 = run_fp32_variant(dp, prob, pos, F, T, torque_mode) if torque_mode == "kernel" else None   # bench.py's fp32_transfer_variant at the size it is timed
    tm = {}
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft", timing=tm, torque_mode=torque_mode)
    if fp32 is not None:
        check_fp32_product("cfg5 (kernel)", fp32[0], fp32[1], U_o, Om_o)
    err = check_product(U, Om, U_o, Om_o)
    print("cfg5 (" + torque_mode + ") whole oracle: stacked rel L2 %.2e, per-particle max %.2e / %.2e, oracle seconds %s" % (
        err, rel_max(U, U_o), rel_max(Om, Om_o), {k: round(v, 1) for k, v in tm.items()}))
