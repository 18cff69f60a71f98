"""GPU parity: the CUDA path (through the C ABI of include/dp.h) against the CPU oracle, element by element, on the
same seeded inputs.  Bar (BASELINE.json north_star): relative L2 <= 1e-10 in fp64.
Stage-level comparisons localise failures (grid after spread, spectra, solve output)."""
import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-10


TOL_MAX = 1e-9      # per-particle bound: max |difference| / max |reference| (one bad particle is invisible in an L2 norm)


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
    dp.load_library()          # fails loudly if the extension is missing
    return dp


def to_dev(*arrs):
    import torch
    return [None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]


def run_gpu(dp, prob, pos, F, T, want_omega=None):
    with dp.Plan(prob, max_particles=len(pos), use_torques=prob.has_torque) as plan:
        dpos, dF, dT = to_dev(pos, F, T)
        U, Om = plan.mobility_apply(dpos, dF, dT, want_omega=want_omega)
        import torch
        torch.cuda.synchronize()
        assert plan.check() == 0
        return U.cpu().numpy(), None if Om is None else Om.cpu().numpy()


def small_monolayer(kind, n, seed):
    """Scaled-down configs 3 / 4: same recipe (area fraction 0.4, heights, drives, w = 6 kernels), fewer particles."""
    if kind == "bw":
        return workloads.monolayer_bw(n=n, seed=seed, name="cfg3-small")
    return workloads.monolayer_slit(n=n, seed=seed, name="cfg4-small")


# ------------------------------------------------------------------------------------------------ stage parity
@pytest.mark.parametrize("dft", ["naive", "fft"])
@pytest.mark.parametrize("case", ["cfg1", "slit-small"])
def test_stage_parity(dp, case, dft):
    """dft = "naive": the oracle's explicit O(n^2) xy DFT sums (the definition north_star names); "fft": its own plain FFT."""
    if case == "cfg1":
        prob, pos, F, T = workloads.config(1)
    else:
        prob, pos, F, T = workloads.random_slit(n=300, L=32.0, nxy=48, nz=48, H=8.0, seed=77, name="slit-small")
    st = {}
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft=dft, stages=st)
    dpos, dF, dT = to_dev(pos, F, T)
    with dp.Plan(prob, max_particles=len(pos), use_torques=prob.has_torque) as plan:
        g = plan.debug_stage(dpos, dF, dT, 1)
        ref = st["f"] if T is None else np.concatenate([st["f"], st["t"]])
        assert rel_l2(g, ref) < 1e-13                                  # only summation order differs
        gh = plan.debug_stage(dpos, dF, dT, 2)
        refh = st["fh"] if T is None else np.concatenate([st["fh"], st["th"]])
        assert rel_l2(gh, refh) < 1e-13
        uh = plan.debug_stage(dpos, dF, dT, 3) * (prob.nx * prob.ny)   # the kernel folds 1/(nx ny) into its output
        refu = st["uh"] if T is None else np.concatenate([st["uh"], st["wh"]])
        nf = refu.shape[0]
        assert rel_l2(uh[:nf], refu) < 1e-11
        # the k = 0 column alone, and the lowest modes alone (worst conditioned)
        assert rel_l2(uh[:nf, :, 0, 0], refu[:, :, 0, 0]) < 1e-11
        assert rel_l2(uh[:nf, :, 0:2, 0:2], refu[:, :, 0:2, 0:2]) < 1e-11
        ur = plan.debug_stage(dpos, dF, dT, 4)
        refr = st["u"] if T is None else np.concatenate([st["u"], st["om"]])
        assert rel_l2(ur[:nf], refr) < 1e-11
        U, Om = plan.mobility_apply(dpos, dF, dT)
        assert rel_l2(U.cpu().numpy(), U_o) < TOL and rel_max(U.cpu().numpy(), U_o) < TOL_MAX
        if T is not None:
            assert rel_l2(Om.cpu().numpy(), Om_o) < TOL and rel_max(Om.cpu().numpy(), Om_o) < TOL_MAX


# ------------------------------------------------------------------------------------------------ full products
@pytest.mark.parametrize("cfg,dft", [(1, "naive"), (1, "fft"), (2, "fft")])
def test_config_parity(dp, cfg, dft):
    """Configs 1 and 2 at full size (configs 3-5: tests/test_gpu_fullsize.py).  Config 1 also with the explicit DFT sums."""
    prob, pos, F, T = workloads.config(cfg)
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft=dft)
    U, Om = run_gpu(dp, prob, pos, F, T)
    err = rel_l2(np.concatenate([U] + ([Om] if Om is not None else []), axis=1),
                 np.concatenate([U_o] + ([Om_o] if Om_o is not None else []), axis=1))
    assert err < TOL, err
    assert rel_l2(U, U_o) < TOL and rel_max(U, U_o) < TOL_MAX
    if Om is not None:
        assert rel_l2(Om, Om_o) < TOL and rel_max(Om, Om_o) < TOL_MAX


@pytest.mark.parametrize("kind,n,seed", [("bw", 3000, 31), ("slit", 2500, 32)])
def test_scaled_monolayer_parity(dp, kind, n, seed):
    """Configs 3 and 4 at reduced N: same recipe; grid not a multiple of the spread tile or of the 32-mode solve tile."""
    prob, pos, F, T = small_monolayer(kind, n, seed)
    assert prob.nx % 16 != 0 or (prob.nx // 2 + 1) % 32 != 0
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft")
    U, Om = run_gpu(dp, prob, pos, F, T)
    assert rel_l2(U, U_o) < TOL and rel_l2(Om, Om_o) < TOL
    assert rel_max(U, U_o) < TOL_MAX and rel_max(Om, Om_o) < TOL_MAX


def test_two_plans_coexist_and_other_devices_work(dp):
    """All device state is per plan (tables, staging buffers, kernel attributes): two plans with different nz alive at once give
    the same results as alone; with >= 2 GPUs visible a plan on device 1 works while device 0 is current."""
    import torch
    pa, posa, Fa, Ta = workloads.random_slit(n=200, L=32.0, nxy=48, nz=32, H=8.0, seed=5, name="A")
    pb, posb, Fb, Tb = workloads.random_bw(n=100, L=32.0, nxy=48, nz=16, H=8.0, seed=6, name="B")
    Ua_o, Oma_o = oracle.mobility_apply(pa, posa, Fa, Ta, dft="fft")
    Ub_o, _ = oracle.mobility_apply(pb, posb, Fb, None, dft="fft")
    with dp.Plan(pa, max_particles=len(posa)) as A, dp.Plan(pb, max_particles=len(posb), use_torques=False) as B:
        for _ in range(2):                                   # interleaved applies
            Ua, Oma = A.mobility_apply(*to_dev(posa, Fa, Ta))
            Ub, _ = B.mobility_apply(*to_dev(posb, Fb))
            Uah, Omah = A.mobility_apply_host(posa, Fa, Ta)
        assert rel_l2(Ua.cpu().numpy(), Ua_o) < TOL and rel_l2(Oma.cpu().numpy(), Oma_o) < TOL
        assert rel_l2(Ub.cpu().numpy(), Ub_o) < TOL and rel_l2(Uah, Ua_o) < TOL
    if torch.cuda.device_count() < 2:
        return
    with dp.Plan(pa, max_particles=len(posa), device=1) as C:
        assert torch.cuda.current_device() == 0
        Uc, Omc = C.mobility_apply_host(posa, Fa, Ta)
        assert torch.cuda.current_device() == 0              # the caller's device is restored
        assert rel_l2(Uc, Ua_o) < TOL and rel_l2(Omc, Oma_o) < TOL
        d1 = [torch.from_numpy(a).to("cuda:1") for a in (posa, Fa, Ta)]
        U1, Om1 = C.mobility_apply(*d1, stream=torch.cuda.current_stream(torch.device("cuda", 1)))
        torch.cuda.synchronize(1)
        assert rel_l2(U1.cpu().numpy(), Ua_o) < TOL


def test_a_later_plan_with_another_grid_size_does_not_disturb_a_live_one(dp):
    """Grid sizes without a static FFT instantiation share the general pass kernels, whose dynamic shared-memory limit is a property of the
    function, not of the plan: a plan created later (smaller or larger grid) must not leave a live plan unable to launch."""
    sizes = (60, 48, 90, 50)
    cases = [workloads.random_bw(n=100, L=nxy * (2.0 / 3.0), nxy=nxy, nz=16, H=8.0, seed=20 + nxy, name="co%d" % nxy) for nxy in sizes]
    refs = [oracle.mobility_apply(pr, pos, F, None, dft="fft")[0] for pr, pos, F, _ in cases]
    plans = []
    try:
        for k, (pr, pos, F, _) in enumerate(cases):
            plans.append(dp.Plan(pr, max_particles=len(pos), use_torques=False))
            for j in range(k + 1):                         # every plan alive so far still works after each creation
                U, _ = plans[j].mobility_apply(*to_dev(cases[j][1], cases[j][2]))
                assert rel_l2(U.cpu().numpy(), refs[j]) < TOL, (k, j)
    finally:
        for pl in plans:
            pl.close()


def test_forces_only_on_a_torque_plan_and_omega_without_torque(dp):
    prob, pos, F, T = workloads.random_slit(n=200, L=32.0, nxy=48, nz=32, H=8.0, seed=5, name="mix")
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, None, want_omega=True, dft="fft")
    U, Om = run_gpu(dp, prob, pos, F, None, want_omega=True)
    assert rel_l2(U, U_o) < TOL and rel_l2(Om, Om_o) < TOL
    U_o2, _ = oracle.mobility_apply(prob, pos, None, T, want_omega=False, dft="fft")
    U2, Om2 = run_gpu(dp, prob, pos, None, T, want_omega=False)
    assert Om2 is None and rel_l2(U2, U_o2) < TOL


# ------------------------------------------------------------------------------------------------ edge cases
def test_edge_cases(dp):
    import torch
    prob, pos, F, T = workloads.random_bw(n=64, L=100 * (2.0 / 3.0) * 0.5, nxy=50, nz=16, H=8.0, seed=9, name="ragged")
    # 50 columns: ragged spread tiles (16 x 8) and a ragged solve tile (26 modes); nz = 16
    pos = pos.copy()
    pos[0, :2] += [7 * prob.Lx, -3 * prob.Ly]        # far outside the primary cell
    pos[1, 2] = 0.0                                  # on the wall: contributes nothing, feels nothing
    pos[2, :2] = [0.0, 0.0]                          # on a grid node
    pos[3, :2] = [prob.Lx - 1e-9, prob.Ly - 1e-9]    # footprint wraps
    U_o, _ = oracle.mobility_apply(prob, pos, F, None, dft="fft")
    U, _ = run_gpu(dp, prob, pos, F, None)
    assert rel_l2(U, U_o) < TOL
    assert np.all(U[1] == 0.0)
    with dp.Plan(prob, max_particles=64, use_torques=False) as plan:
        # n = 0 is a no-op
        e = torch.empty((0, 3), dtype=torch.float64, device="cuda")
        U0, _ = plan.mobility_apply(e, e)
        assert U0.shape == (0, 3)
        # out-of-domain particles: flagged, contribute nothing, get zero
        bad = pos.copy()
        bad[5, 2] = -0.1
        bad[6, 2] = prob.H - 0.5                      # bottom wall: kernel would cross the open top
        dpos, dF = to_dev(bad, F)
        Ub, _ = plan.mobility_apply(dpos, dF)
        torch.cuda.synchronize()
        assert plan.check() == -5
        keep = np.ones(len(pos), bool); keep[[5, 6]] = False
        U_ref, _ = oracle.mobility_apply(prob, bad[keep], F[keep], None, dft="fft")
        Ub = Ub.cpu().numpy()
        assert np.all(Ub[[5, 6]] == 0.0) and rel_l2(Ub[keep], U_ref) < TOL
        # both inputs missing -> error, not a crash
        with pytest.raises(dp.DPError):
            plan.mobility_apply(dpos, None, None)
        # the plan is reusable and repeatable (bin order may differ: <= 1e-13, reading G16)
        U1, _ = plan.mobility_apply(*to_dev(pos, F))
        U2, _ = plan.mobility_apply(*to_dev(pos, F))
        assert rel_l2(U1.cpu().numpy(), U2.cpu().numpy()) < 1e-13


@pytest.mark.parametrize("mode", ["fourier", "kernel", "forces"])
def test_clustered_particles_take_both_spreading_paths(dp, mode):
    """Spreading runs per-tile survivor lists through a pipelined kernel and leaves tiles whose list does not fit a staged chunk (20 particles
    with kernel-derivative torques, 40 otherwise) to the culling kernel: a cluster of 300 particles inside a 6 x 6 patch (every tile it
    touches overflows, hundreds of survivors per tile = several chunks) plus a dilute background (lists of 0..5) exercises both, and the
    interpolation of many particles from the same columns.  Result against the oracle."""
    import dataclasses
    prob, pos, F, T = workloads.random_slit(n=700, L=40.0, nxy=60, nz=24, H=8.0, seed=4242, name="cluster")
    rng = np.random.default_rng(4243)
    pos = pos.copy()
    pos[:300, 0] = 11.0 + 6.0 * rng.random(300)
    pos[:300, 1] = 23.0 + 6.0 * rng.random(300)
    if mode == "forces":
        prob = dataclasses.replace(prob, has_torque=False); T = None
    tm = 1 if mode == "kernel" else 0
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft", torque_mode="kernel" if tm else "fourier")
    with dp.Plan(prob, max_particles=len(pos), use_torques=T is not None, torque_mode=tm) as plan:
        U, Om = plan.mobility_apply(*to_dev(pos, F, T))
        assert plan.check() == 0
    assert rel_l2(U.cpu().numpy(), U_o) < TOL and rel_max(U.cpu().numpy(), U_o) < TOL_MAX
    if T is not None:
        assert rel_l2(Om.cpu().numpy(), Om_o) < TOL and rel_max(Om.cpu().numpy(), Om_o) < TOL_MAX


def test_host_entry_point_matches_device_entry_point(dp):
    prob, pos, F, T = workloads.random_slit(n=500, L=32.0, nxy=48, nz=32, H=8.0, seed=12, name="host")
    with dp.Plan(prob, max_particles=len(pos)) as plan:
        Uh, Omh = plan.mobility_apply_host(pos, F, T)
        U, Om = plan.mobility_apply(*to_dev(pos, F, T))
        assert rel_l2(Uh, U.cpu().numpy()) < 1e-13 and rel_l2(Omh, Om.cpu().numpy()) < 1e-13


def test_create_rejects_bad_parameters(dp):
    prob, *_ = workloads.config(1)
    import dataclasses
    for bad in (dict(nz=7), dict(nz=31), dict(nx=49), dict(w=3), dict(eta=0.0), dict(Ly=prob.Ly * 1.01), dict(nx=16, ny=16)):
        with pytest.raises(dp.DPError):
            dp.Plan(dataclasses.replace(prob, **bad), max_particles=8)


# ------------------------------------------------------------------------------------------------ xy FFT passes
def _rfft2(a):
    return np.fft.rfft2(a, axes=(-2, -1))


@pytest.mark.parametrize("kind,nxy,nz,n", [("bw", 216, 32, 1500), ("slit", 240, 48, 1500), ("bw", 50, 16, 64), ("bw", 1080, 16, 3000)])
def test_own_fft_passes_match_the_dft_and_cufft(dp, kind, nxy, nz, n):
    """The library's own xy FFT passes (transposed, digit-reversed half spectrum) against the unnormalised DFT definition
    (numpy.fft.rfft2, the primitive the oracle's DFT is pinned to) and against the cuFFT backend; nxy = 50 cannot be
    factored into the compiled radices' batch shapes differently: it exercises the general kernels, 1080 the static ones."""
    L = nxy * (2.0 / 3.0)
    mk = workloads.random_bw if kind == "bw" else workloads.random_slit
    prob, pos, F, T = mk(n=n, L=L, nxy=nxy, nz=nz, H=8.0, seed=41, name="fft")
    if nxy >= 1000:
        T = None                                                     # three fields are enough at this size
    dpos, dF, dT = to_dev(pos, F, T)
    res = {}
    for backend in (0, 1):
        with dp.Plan(prob, max_particles=n, use_torques=T is not None, fft_backend=backend) as plan:
            assert plan.fft_backend() == ("own" if backend == 0 else "cufft")
            g = plan.debug_stage(dpos, dF, dT, 1)
            gh = plan.debug_stage(dpos, dF, dT, 2)
            assert rel_l2(gh, _rfft2(g)) < 1e-14
            uh = plan.debug_stage(dpos, dF, dT, 3)
            ur = plan.debug_stage(dpos, dF, dT, 4)
            nf = 6 if T is not None else 3
            back = np.fft.irfft2(uh[:nf], s=(prob.ny, prob.nx), axes=(-2, -1)) * (prob.nx * prob.ny)
            assert rel_l2(ur[:nf], back) < 1e-13
            U, Om = plan.mobility_apply(dpos, dF, dT)
            res[backend] = U.cpu().numpy()
    assert rel_l2(res[0], res[1]) < 1e-13


def test_unsupported_fft_size_falls_back_to_cufft(dp):
    prob, pos, F, T = workloads.random_bw(n=64, L=28 * (2.0 / 3.0), nxy=28, nz=16, H=8.0, seed=3, name="seven")   # 28 = 4 * 7
    with dp.Plan(prob, max_particles=64, use_torques=False) as plan:
        assert plan.fft_backend() == "cufft"
        U_o, _ = oracle.mobility_apply(prob, pos, F, None, dft="fft")
        U, _ = plan.mobility_apply(*to_dev(pos, F))
        assert rel_l2(U.cpu().numpy(), U_o) < TOL


def test_full_size_fft_passes_on_sampled_planes_and_backends_agree(dp):
    """BASELINE config 5 (4320 x 4320 x 32, N = 1,048,576, the configuration bench.py times, same launch configuration):
    the oracle cannot finish this size, so (i) sampled planes of the forward spectrum are compared with numpy's rfft2 of
    the spread grid, (ii) the whole product is compared between the own FFT passes and the cuFFT backend, and (iii) the
    properties that hold at any size are checked: U = 0 for a particle on the wall, and the product is linear."""
    import torch
    prob, pos, F, T = workloads.config(5)
    n = len(pos)
    pos = pos.copy()
    pos[7, 2] = 0.0
    dpos, dF, dT = to_dev(pos, F, T)
    with dp.Plan(prob, max_particles=n, use_torques=True, fft_backend=0) as plan:
        assert plan.fft_backend() == "own"
        U, Om = plan.mobility_apply(dpos, dF, dT)
        U2, Om2 = plan.mobility_apply(dpos, 2.0 * dF, 2.0 * dT)
        torch.cuda.synchronize()
        assert plan.check() == 0
        U, Om, U2, Om2 = (t.cpu().numpy() for t in (U, Om, U2, Om2))
        assert np.all(U[7] == 0.0) and np.all(Om[7] == 0.0)
        assert rel_l2(U2, 2.0 * U) < 1e-13 and rel_l2(Om2, 2.0 * Om) < 1e-13
        # sampled planes of the forward transform of field 0 (f_x), near the wall (only field 0 is copied to the host: 4.8 GB)
        import ctypes
        L = dp.load_library()
        st = torch.cuda.current_stream()
        ptr = lambda t: ctypes.c_void_p(t.data_ptr())
        for stage, which in ((1, 0), (2, 1)):
            rc = L.dp_debug_run_stage(plan._h, n, ptr(dpos), ptr(dF), ptr(dT), stage, ctypes.c_void_p(st.cuda_stream))
            assert rc == 0
            torch.cuda.synchronize()
            if stage == 1:
                planes = {}
                real = np.empty((1, prob.nz, prob.ny, prob.nx))
                assert L.dp_copy_buffer_to_host(plan._h, 0, real.ctypes.data_as(ctypes.c_void_p), real.nbytes) == 0
                for f, l in ((0, prob.nz - 3), (0, prob.nz - 6)):
                    assert np.abs(real[f, l]).max() > 0
                    planes[(f, l)] = _rfft2(real[f, l])
                del real
            else:
                pitch = int(L.dp_complex_row_pitch(plan._h))
                spec = np.empty((1, prob.nz, prob.ny, pitch), dtype=np.complex128)
                assert L.dp_copy_buffer_to_host(plan._h, 1, spec.ctypes.data_as(ctypes.c_void_p), spec.nbytes) == 0
                for (f, l), ref in planes.items():
                    assert rel_l2(spec[f, l, :, : prob.nx // 2 + 1], ref) < 1e-14
                del spec
    with dp.Plan(prob, max_particles=n, use_torques=True, fft_backend=1) as plan:
        Uc, Omc = plan.mobility_apply(dpos, dF, dT)
        torch.cuda.synchronize()
        assert rel_l2(Uc.cpu().numpy(), U) < 1e-12 and rel_l2(Omc.cpu().numpy(), Om) < 1e-12


# ------------------------------------------------------------------------------------------------ fp32 transfer variant
@pytest.mark.parametrize("case", ["cfg1", "cfg2", "bw-mono", "slit-mono"])
def test_fp32_transfer_variant_matches_the_oracle_to_1e5(dp, case):
    """north_star: the optional fp32 spread/interpolate variant (fp32 accumulation and fp32 real-space grids, fp64 transforms
    and solves) must match the oracle to a relative L2 error <= 1e-5."""
    if case == "cfg1":
        prob, pos, F, T = workloads.config(1)
    elif case == "cfg2":
        prob, pos, F, T = workloads.config(2)
    elif case == "bw-mono":
        prob, pos, F, T = small_monolayer("bw", 3000, 31)
    else:
        prob, pos, F, T = small_monolayer("slit", 2500, 32)
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft")
    with dp.Plan(prob, max_particles=len(pos), use_torques=prob.has_torque, transfer_fp32=True) as plan:
        U, Om = plan.mobility_apply(*to_dev(pos, F, T))
        import torch
        torch.cuda.synchronize()
        assert plan.check() == 0
        e = rel_l2(U.cpu().numpy(), U_o)
        assert 1e-9 < e < 1e-5, e                       # really fp32 (not silently fp64), and within the bar
        if Om is not None:
            assert rel_l2(Om.cpu().numpy(), Om_o) < 1e-5
        # the spread grid handed out by the test hook is the fp32 grid widened to doubles
        g = plan.debug_stage(*to_dev(pos, F, T), 1)
        st = {}
        oracle.mobility_apply(prob, pos, F, T, dft="fft", stages=st)
        ref = st["f"] if T is None else np.concatenate([st["f"], st["t"]])
        assert 1e-9 < rel_l2(g, ref) < 1e-6
    # the variant needs the own FFT passes
    with pytest.raises(dp.DPError):
        dp.Plan(prob, max_particles=len(pos), use_torques=prob.has_torque, transfer_fp32=True, fft_backend=1)


# ------------------------------------------------------------------------------------------------ zero planes
def test_skipping_the_zero_planes_is_exact(dp):
    """Planes above every footprint hold no force; the product skips their spreading stores, forward FFT passes and solve
    loads.  Skipping changes no arithmetic: the result equals the dense-plane product to the run-to-run noise of the spreading order
    and the oracle to 1e-10."""
    import torch
    prob, pos, F, T = small_monolayer("bw", 3000, 31)          # heights 1 + Exp(0.5): the top of the z grid stays empty
    dpos, dF, dT = to_dev(pos, F, T)
    out = {}
    for dense in (False, True):
        with dp.Plan(prob, max_particles=len(pos), use_torques=True, dense_planes=dense) as plan:
            # stale data in the buffers must not matter: run a different product first
            plan.mobility_apply(dpos, 3.0 * dF, dT)
            U, Om = plan.mobility_apply(dpos, dF, dT)
            torch.cuda.synchronize()
            zp = plan.zero_planes()
            assert (zp == 0) if dense else (3 <= zp < prob.nz), zp
            out[dense] = (U.cpu().numpy(), Om.cpu().numpy())
    # same arithmetic on the same values; only the bin order of spreading differs from run to run (<= 1e-13, reading G16)
    assert rel_l2(out[False][0], out[True][0]) < 1e-13 and rel_l2(out[False][1], out[True][1]) < 1e-13
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft")
    assert rel_l2(out[False][0], U_o) < TOL and rel_l2(out[False][1], Om_o) < TOL
    # a slit with particles up to the top wall has no empty plane
    prob, pos, F, T = small_monolayer("slit", 2500, 32)
    with dp.Plan(prob, max_particles=len(pos), use_torques=True) as plan:
        plan.mobility_apply(*to_dev(pos, F, T))
        assert plan.zero_planes() == 0


# ------------------------------------------------------------------------------------------------ kernel-derivative torques
@pytest.mark.parametrize("case", ["slit", "bw-monolayer", "cfg2"])
def test_kernel_derivative_torque_mode_matches_the_oracle(dp, case):
    """dp_params.torque_mode = 1 (footnotes 47-48): torques spread with the ES kernel's derivative into the force field,
    Omega gathered from u itself; three grid fields each way.  Against the oracle's own kernel-derivative path."""
    import dataclasses
    if case == "slit":
        prob, pos, F, T = workloads.random_slit(n=300, L=32.0, nxy=48, nz=48, H=8.0, seed=78, name="slit-small")
        pos = pos.copy(); pos[:5, 2] = [0.0, 0.2, 7.9, 8.0, 4.0]            # on and next to both walls
    elif case == "bw-monolayer":
        prob, pos, F, T = small_monolayer("bw", 3000, 41)
    else:
        prob, pos, F, T = workloads.config(2)
    st = {}
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft", torque_mode="kernel", stages=st)
    dpos, dF, dT = to_dev(pos, F, T)
    with dp.Plan(prob, max_particles=len(pos), use_torques=True, torque_mode=1) as plan:
        assert plan.fields == 3
        g = plan.debug_stage(dpos, dF, dT, 1)
        assert g.shape[0] == 3 and rel_l2(g, st["f"]) < 1e-13 and rel_max(g, st["f"]) < 1e-12
        ur = plan.debug_stage(dpos, dF, dT, 4)
        assert rel_l2(ur, st["u"]) < 1e-11
        U, Om = plan.mobility_apply(dpos, dF, dT)
        U, Om = U.cpu().numpy(), Om.cpu().numpy()
        assert plan.check() == 0
        assert rel_l2(np.concatenate([U, Om], axis=1), np.concatenate([U_o, Om_o], axis=1)) < TOL
        assert rel_l2(U, U_o) < TOL and rel_max(U, U_o) < TOL_MAX
        assert rel_l2(Om, Om_o) < TOL and rel_max(Om, Om_o) < TOL_MAX
        # forces only on the same plan; torques only; Omega not wanted
        U1, _ = plan.mobility_apply(dpos, dF, None, want_omega=False)
        U1_o, _ = oracle.mobility_apply(prob, pos, F, None, dft="fft", torque_mode="kernel")
        assert rel_l2(U1.cpu().numpy(), U1_o) < TOL
        U2, Om2 = plan.mobility_apply(dpos, None, dT)
        U2_o, Om2_o = oracle.mobility_apply(prob, pos, None, T, dft="fft", torque_mode="kernel")
        assert rel_l2(U2.cpu().numpy(), U2_o) < TOL and rel_l2(Om2.cpu().numpy(), Om2_o) < TOL
        Uh, Omh = plan.mobility_apply_host(pos, F, T)
        assert rel_l2(Uh, U_o) < TOL and rel_l2(Omh, Om_o) < TOL
    # and the two ways agree with each other to the method's 2-3 digits, not to roundoff
    with dp.Plan(prob, max_particles=len(pos), use_torques=True, torque_mode=0) as plan0:
        U0, Om0 = plan0.mobility_apply(dpos, dF, dT)
    assert 1e-8 < rel_l2(Om, Om0.cpu().numpy()) < 5e-2 and rel_l2(U, U0.cpu().numpy()) < 5e-2


def test_kernel_derivative_mode_fp32_transfer_variant(dp):
    prob, pos, F, T = small_monolayer("bw", 3000, 43)
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft", torque_mode="kernel")
    with dp.Plan(prob, max_particles=len(pos), use_torques=True, torque_mode=1, transfer_fp32=True) as plan:
        U, Om = plan.mobility_apply(*to_dev(pos, F, T))
    eU, eO = rel_l2(U.cpu().numpy(), U_o), rel_l2(Om.cpu().numpy(), Om_o)
    assert 1e-9 < eU < 1e-5 and 1e-9 < eO < 1e-5, (eU, eO)


# ------------------------------------------------------------------------------------------------ other Chebyshev sizes and kernel widths
@pytest.mark.parametrize("nz,w,wall", [(19, 4, "bw"), (26, 6, "bw"), (24, 5, "slit"), (40, 8, "slit"), (64, 7, "bw"), (16, 4, "slit")])
def test_every_compiled_chebyshev_size_and_kernel_width(dp, nz, w, wall):
    """The paper's own performance grids use Nz = 19 (monopole only, m = 4) and Nz = 26 (Table III): every size in
    dp_supported_nz (odd ones included: the middle Chebyshev node pairs with itself) and every width 4..8, against the oracle."""
    import dataclasses
    assert nz in dp.supported_nz()
    beta_M = {4: 4 * 1.785, 5: 5 * 1.886, 6: 6 * 1.327, 7: 7 * 1.5, 8: 8 * 1.4}[w]
    beta_D = {4: 4 * 2.4, 5: 5 * 2.232, 6: 6 * 2.216, 7: 7 * 2.1, 8: 8 * 2.0}[w]
    if wall == "bw":
        prob, pos, F, _ = workloads.random_bw(n=150, L=40.0, nxy=50, nz=nz, H=9.0, zlo=0.0, zhi=9.0 - 0.5 * w * 0.8, seed=500 + nz, name="nz")
        T = np.random.default_rng(nz).standard_normal(F.shape)
    else:
        prob, pos, F, T = workloads.random_slit(n=150, L=40.0, nxy=50, nz=nz, H=9.0, margin=0.0, seed=500 + nz, name="nz")
    prob = dataclasses.replace(prob, w=w, beta_M=beta_M, beta_D=beta_D, has_torque=True)
    for mode, name in ((0, "fourier"), (1, "kernel")):
        U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft", torque_mode=name)
        with dp.Plan(prob, max_particles=len(pos), use_torques=True, torque_mode=mode) as plan:
            U, Om = plan.mobility_apply(*to_dev(pos, F, T))
            assert plan.check() == 0
        assert rel_l2(U.cpu().numpy(), U_o) < TOL and rel_l2(Om.cpu().numpy(), Om_o) < TOL, (mode, nz, w)
        assert rel_max(U.cpu().numpy(), U_o) < TOL_MAX and rel_max(Om.cpu().numpy(), Om_o) < TOL_MAX


# ------------------------------------------------------------------------------------------------ the two solve kernels
@pytest.mark.parametrize("case", ["bw-forces", "slit-forces-nz26", "slit-kernel-torques-slip", "bw-kernel-torques-ragged-nz19"])
def test_both_solve_kernels_match_the_oracle_and_each_other(dp, case):
    """Products with three grid fields each way run steps 2(z)-6 in the warp-pair kernel (solve_pair.cu) by default;
    dp_params.solve_kernel = 1 keeps the tile kernel (solve.cu).  Both solve the oracle's discrete problem: each <= 1e-10 from the
    oracle, and they agree with one another to roundoff (the nodal correction equals the coefficient-space one)."""
    import dataclasses
    if case == "bw-forces":
        prob, pos, F, T = workloads.random_bw(n=300, L=40.0, nxy=60, nz=32, H=9.0, seed=811, name=case)
        T = None; mode = 0
    elif case == "slit-forces-nz26":
        prob, pos, F, T = workloads.random_slit(n=300, L=36.0, nxy=54, nz=26, H=8.0, seed=812, name=case)
        prob = dataclasses.replace(prob, has_torque=False); T = None; mode = 0
    elif case == "slit-kernel-torques-slip":
        prob, pos, F, T = workloads.random_slit(n=300, L=32.0, nxy=48, nz=40, H=8.0, seed=813, name=case)
        prob = dataclasses.replace(prob, slip_0=0.3, slip_H=0.7); mode = 1
    else:
        prob, pos, F, _ = workloads.random_bw(n=200, L=40.0, nxy=50, nz=19, H=9.0, zlo=0.0, zhi=6.0, seed=814, name=case)   # 50 = 3 tiles of 16 + 2
        T = np.random.default_rng(814).standard_normal(F.shape); prob = dataclasses.replace(prob, has_torque=True, beta_M=6 * 1.327, beta_D=6 * 2.216); mode = 1
    use_t = T is not None
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft", torque_mode="kernel" if mode else "fourier")
    out = {}
    for sk in (0, 1):
        with dp.Plan(prob, max_particles=len(pos), use_torques=use_t, torque_mode=mode, solve_kernel=sk) as plan:
            U, Om = plan.mobility_apply(*to_dev(pos, F, T))
            assert plan.check() == 0
            out[sk] = (U.cpu().numpy(), None if Om is None else Om.cpu().numpy())
        assert rel_l2(out[sk][0], U_o) < TOL and rel_max(out[sk][0], U_o) < TOL_MAX, (case, sk)
        if use_t:
            assert rel_l2(out[sk][1], Om_o) < TOL and rel_max(out[sk][1], Om_o) < TOL_MAX, (case, sk)
    assert rel_l2(out[0][0], out[1][0]) < 1e-12
    if use_t:
        assert rel_l2(out[0][1], out[1][1]) < 1e-12


# ------------------------------------------------------------------------------------------------ Lanczos square root
@pytest.mark.parametrize("with_torque,mode", [(False, 0), (True, 1), (True, 0)])
def test_lanczos_square_root_matches_the_oracle_iteration(dp, with_torque, mode):
    """dp_lanczos_sqrt (Sec. V B) against the oracle's Lanczos driven by the oracle's own mobility product: same
    iteration count, same eps_n history (Fig. 11's quantity), same g."""
    prob, pos, F, T = small_monolayer("bw", 400, 51)
    n = len(pos)
    rng = np.random.default_rng(9)
    WF = rng.standard_normal((n, 3))
    WT = rng.standard_normal((n, 3)) if with_torque else None
    name = "kernel" if mode else "fourier"

    def apply(v):
        if with_torque:
            U, Om = oracle.mobility_apply(prob, pos, v[:3 * n].reshape(n, 3), v[3 * n:].reshape(n, 3), dft="fft", torque_mode=name)
            return np.concatenate([U.ravel(), Om.ravel()])
        U, _ = oracle.mobility_apply(prob, pos, v.reshape(n, 3), None, dft="fft")
        return U.ravel()

    W = np.concatenate([WF.ravel(), WT.ravel()]) if with_torque else WF.ravel()
    g_o, its_o, eps_o = oracle.lanczos_sqrt(apply, W, tol=1e-4, max_iter=40)
    with dp.Plan(prob, max_particles=n, use_torques=True, torque_mode=mode) as plan:
        gU, gO, its, eps = plan.lanczos_sqrt(*to_dev(pos, WF, WT), tol=1e-4, max_iter=40)
    g = np.concatenate([gU.cpu().numpy().ravel()] + ([gO.cpu().numpy().ravel()] if with_torque else []))
    assert its == its_o and len(eps) == len(eps_o)
    assert np.allclose(eps, eps_o, rtol=1e-5)
    assert rel_l2(g, g_o) < 1e-8
    assert its < 40                                             # converged before max_iter


def test_lanczos_on_the_fp32_transfer_variant_converges_like_the_fp64_run(dp):
    """Fig. 12's caption: above ~1e-6 the convergence of the Lanczos iteration is not affected by single vs double
    precision.  dp_lanczos_sqrt on a transfer_fp32 plan against the fp64 plan: same number of products at the paper's working tolerance
    (1e-3) and at 1e-4 (measured: 17 and 38 at both precisions), within one product at 1e-5 (which may hit the 64-product limit of the entry point),
    eps_n histories that agree wherever eps_n > 1e-4 (measured: to 8e-3 relative), and the same g to the variant's accuracy (measured: 1e-7)."""
    prob, pos, F, T = small_monolayer("bw", 2000, 53)
    n = len(pos)
    rng = np.random.default_rng(10)
    WF, WT = rng.standard_normal((n, 3)), rng.standard_normal((n, 3))
    out = {}
    for f32 in (False, True):
        with dp.Plan(prob, max_particles=n, use_torques=True, torque_mode=1, transfer_fp32=f32) as plan:
            for tol in (1e-3, 1e-4, 1e-5):
                gU, gO, its, eps = plan.lanczos_sqrt(*to_dev(pos, WF, WT), tol=tol, max_iter=64)
                out[(f32, tol)] = (np.concatenate([gU.cpu().numpy().ravel(), gO.cpu().numpy().ravel()]), its, np.array(eps))
    for tol in (1e-3, 1e-4, 1e-5):
        g64, its64, eps64 = out[(False, tol)]
        g32, its32, eps32 = out[(True, tol)]
        m = min(len(eps64), len(eps32))
        big = eps64[:m] > 1e-4
        print("lanczos tol %.0e: products fp64 %d / fp32 %d, max rel eps difference above 1e-4: %.2e, g rel L2 %.2e" % (
            tol, its64, its32, float(np.abs(eps32[:m][big] / eps64[:m][big] - 1).max()) if big.any() else 0.0, rel_l2(g32, g64)))
        if tol >= 1e-4:
            assert its64 < 64 and its32 == its64                # converged, and after the same number of products
        else:
            assert abs(its32 - its64) <= 1
        assert np.allclose(eps32[:m][big], eps64[:m][big], rtol=2e-2)
        assert rel_l2(g32, g64) < max(1e-5, 3 * tol)


def test_lanczos_refuses_a_plan_whose_product_is_affine(dp):
    """With moving walls U = M F + (wall-driven flow): not a linear SPD operator, so M^{1/2} W has no meaning (dp.h)."""
    import dataclasses
    prob, pos, F, T = small_monolayer("bw", 100, 54)
    with dp.Plan(dataclasses.replace(prob, uwall_0=(0.5, 0.0)), max_particles=len(pos)) as plan:
        with pytest.raises(dp.DPError, match="wall velocity"):
            plan.lanczos_sqrt(*to_dev(pos, F, T), tol=1e-3, max_iter=10)


# ------------------------------------------------------------------------------------------------ partial slip, moving walls
@pytest.mark.parametrize("case", ["slit-slip", "slit-slip-top-only", "slit-moving-walls", "bw-moving-wall", "slit-all-kernel-mode"])
def test_partial_slip_and_moving_walls_match_the_oracle(dp, case):
    """Appendix A: slip lengths l_0, l_H in the slit ((A8), (A12)) and uniform wall velocities (eqs 27, 46, 52),
    against the oracle's general 8 x 8 correction solve and its k = 0 system with slip rows."""
    import dataclasses
    mode = 0
    if case.startswith("slit"):
        prob, pos, F, T = workloads.random_slit(n=300, L=32.0, nxy=48, nz=48, H=8.0, seed=91, name=case)
        pos = pos.copy(); pos[:4, 2] = [0.0, 0.3, 7.8, 8.0]
        if case == "slit-slip":
            prob = dataclasses.replace(prob, slip_0=0.7, slip_H=0.25)
        elif case == "slit-slip-top-only":
            prob = dataclasses.replace(prob, slip_H=3.0)
        elif case == "slit-moving-walls":
            prob = dataclasses.replace(prob, uwall_0=(0.3, -0.1), uwall_H=(-1.2, 0.4))
        else:
            prob = dataclasses.replace(prob, slip_0=0.4, slip_H=1.1, uwall_0=(0.3, -0.1), uwall_H=(-1.2, 0.4))
            mode = 1
    else:
        prob, pos, F, T = small_monolayer("bw", 1500, 93)
        prob = dataclasses.replace(prob, uwall_0=(0.8, 0.5))
    U_o, Om_o = oracle.mobility_apply(prob, pos, F, T, dft="fft", torque_mode="kernel" if mode else "fourier")
    with dp.Plan(prob, max_particles=len(pos), use_torques=True, torque_mode=mode) as plan:
        U, Om = plan.mobility_apply(*to_dev(pos, F, T))
        assert plan.check() == 0
    U, Om = U.cpu().numpy(), Om.cpu().numpy()
    assert rel_l2(U, U_o) < TOL and rel_max(U, U_o) < TOL_MAX
    assert rel_l2(Om, Om_o) < TOL and rel_max(Om, Om_o) < TOL_MAX
    # the wall data really matter: the no-slip, resting-wall product differs
    base = dataclasses.replace(prob, slip_0=0.0, slip_H=0.0, uwall_0=(0.0, 0.0), uwall_H=(0.0, 0.0))
    with dp.Plan(base, max_particles=len(pos), use_torques=True, torque_mode=mode) as plan0:
        U0, _ = plan0.mobility_apply(*to_dev(pos, F, T))
    assert rel_l2(U, U0.cpu().numpy()) > 1e-3


def test_wall_data_that_the_paper_gives_no_solution_for_are_rejected(dp):
    import dataclasses
    prob, pos, F, T = small_monolayer("bw", 100, 94)
    for bad in (dict(slip_0=0.1), dict(slip_H=0.1), dict(uwall_H=(0.1, 0.0))):
        with pytest.raises(dp.DPError):
            dp.Plan(dataclasses.replace(prob, **bad), max_particles=len(pos))
    probS, *_ = workloads.random_slit(n=10, L=32.0, nxy=48, nz=32, H=8.0, seed=1, name="s")
    with pytest.raises(dp.DPError):
        dp.Plan(dataclasses.replace(probS, slip_0=-0.1), max_particles=10)
