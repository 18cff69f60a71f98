"""ctypes binding of include/dp.h — same names, argument marshalling only."""
from __future__ import annotations

import ctypes
import os

import numpy as np

BOTTOM_WALL = 0
SLIT = 1

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBNAME = os.path.join(_HERE, "libdpstokes.so")

# every symbol include/dp.h declares
EXPORTS = ["dp_create", "dp_mobility_apply", "dp_mobility_apply_host", "dp_lanczos_sqrt", "dp_bin_particles_static", "dp_copy_bins_to_host", "dp_check", "dp_effective_radius", "dp_set_profiling", "dp_stage_ms", "dp_fft_pass_ms",
           "dp_debug_run_stage", "dp_buffer_bytes", "dp_copy_buffer_to_host", "dp_copy_plane_to_host", "dp_complex_row_pitch", "dp_zero_planes", "dp_fft_backend", "dp_solve_kernel", "dp_es_norm", "dp_es_radius_over_h",
           "dp_es_dphi_cut", "dp_supported_nz", "dp_device_bytes", "dp_strerror", "dp_last_error", "dp_destroy"]


class DPError(RuntimeError):
    pass


class dp_params(ctypes.Structure):
    _fields_ = [("wall_mode", ctypes.c_int), ("Lx", ctypes.c_double), ("Ly", ctypes.c_double), ("H", ctypes.c_double),
                ("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int), ("w", ctypes.c_int),
                ("beta_M", ctypes.c_double), ("beta_D", ctypes.c_double), ("a", ctypes.c_double), ("eta", ctypes.c_double),
                ("max_particles", ctypes.c_int), ("transfer_fp32", ctypes.c_int), ("device", ctypes.c_int),
                # extensions beyond SURVEY.md §8(b)
                ("use_torques", ctypes.c_int), ("fft_backend", ctypes.c_int), ("dense_planes", ctypes.c_int), ("torque_mode", ctypes.c_int),
                ("slip_0", ctypes.c_double), ("slip_H", ctypes.c_double), ("uwall_0", ctypes.c_double * 2), ("uwall_H", ctypes.c_double * 2),
                ("solve_kernel", ctypes.c_int)]


_lib = None


def library_path() -> str:
    return _LIBNAME


def load_library():
    """Load libdpstokes.so (built in-tree by ``build.py`` / ``__graft_entry__.build()``).  No fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIBNAME):
        raise DPError("CUDA library %s is missing: run `python -m paper_2210_01837_b200.build` "
                      "(or __graft_entry__.build()); there is no CPU fallback" % _LIBNAME)
    L = ctypes.CDLL(_LIBNAME)
    vp, i, d, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    L.dp_create.argtypes = [ctypes.POINTER(dp_params), ctypes.POINTER(vp)]
    L.dp_create.restype = i
    L.dp_mobility_apply.argtypes = [vp, i, vp, vp, vp, vp, vp, vp]
    L.dp_mobility_apply.restype = i
    L.dp_mobility_apply_host.argtypes = [vp, i, vp, vp, vp, vp, vp]
    L.dp_mobility_apply_host.restype = i
    L.dp_lanczos_sqrt.argtypes = [vp, i, vp, vp, vp, vp, vp, d, i, ctypes.POINTER(i), ctypes.POINTER(d), vp]
    L.dp_lanczos_sqrt.restype = i
    L.dp_bin_particles_static.argtypes = [ctypes.POINTER(dp_params), i, vp, vp, vp, vp]
    L.dp_bin_particles_static.restype = i
    L.dp_copy_bins_to_host.argtypes = [vp, i, vp, vp]
    L.dp_copy_bins_to_host.restype = i
    L.dp_check.argtypes = [vp]
    L.dp_check.restype = i
    L.dp_set_profiling.argtypes = [vp, i]
    L.dp_set_profiling.restype = i
    L.dp_stage_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    L.dp_stage_ms.restype = i
    L.dp_fft_pass_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    L.dp_fft_pass_ms.restype = i
    L.dp_debug_run_stage.argtypes = [vp, i, vp, vp, vp, i, vp]
    L.dp_debug_run_stage.restype = i
    L.dp_buffer_bytes.argtypes = [vp, i]
    L.dp_buffer_bytes.restype = sz
    L.dp_copy_buffer_to_host.argtypes = [vp, i, vp, sz]
    L.dp_copy_buffer_to_host.restype = i
    L.dp_copy_plane_to_host.argtypes = [vp, i, i, i, vp, sz]
    L.dp_copy_plane_to_host.restype = i
    L.dp_effective_radius.argtypes = [vp, i]
    L.dp_effective_radius.restype = d
    L.dp_complex_row_pitch.argtypes = [vp]
    L.dp_complex_row_pitch.restype = i
    L.dp_zero_planes.argtypes = [vp]
    L.dp_zero_planes.restype = i
    L.dp_fft_backend.argtypes = [vp]
    L.dp_fft_backend.restype = i
    L.dp_solve_kernel.argtypes = [vp]
    L.dp_solve_kernel.restype = i
    L.dp_es_norm.argtypes = [d, d]
    L.dp_es_norm.restype = d
    L.dp_es_radius_over_h.argtypes = [i, d, i]
    L.dp_es_radius_over_h.restype = d
    L.dp_es_dphi_cut.argtypes = [d]
    L.dp_es_dphi_cut.restype = d
    L.dp_supported_nz.argtypes = [ctypes.POINTER(i), i]
    L.dp_supported_nz.restype = i
    L.dp_device_bytes.argtypes = [vp]
    L.dp_device_bytes.restype = sz
    L.dp_strerror.argtypes = [i]
    L.dp_strerror.restype = ctypes.c_char_p
    L.dp_last_error.argtypes = [vp]
    L.dp_last_error.restype = ctypes.c_char_p
    L.dp_destroy.argtypes = [vp]
    L.dp_destroy.restype = i
    _lib = L
    return L


def exported_symbols():
    L = load_library()
    return [s for s in EXPORTS if hasattr(L, s)]


def es_norm(alpha: float, beta: float) -> float:
    return float(load_library().dp_es_norm(alpha, beta))


def es_dphi_cut(beta: float) -> float:
    return float(load_library().dp_es_dphi_cut(beta))


def supported_nz():
    buf = (ctypes.c_int * 16)()
    n = load_library().dp_supported_nz(buf, 16)
    return [int(buf[k]) for k in range(n)]


BIN_TILE_X, BIN_TILE_Y = 16, 4                                      # DP_BIN_TILE_X, DP_BIN_TILE_Y
STATIC_BIN_MAX_PARTICLES, STATIC_BIN_MAX_TILES = 262144, 131072     # DP_STATIC_BIN_MAX_PARTICLES, DP_STATIC_BIN_MAX_TILES
ETOOBIG = -6


def bin_particles_static(params: dp_params, pos, perm=None, tile_start=None, stream=None):
    """dp_bin_particles_static: the product's counting sort of the particles by xy tile for callers that may not allocate device
    memory (see include/dp.h: its work arrays are a fixed array inside the library, at most 262,144 particles and 131,072 tiles).
    ``pos`` float64 CUDA tensor [n,3]; ``perm`` [n] and ``tile_start`` [tiles+1] int32 CUDA tensors are the caller's outputs (made
    here with torch only when not given — pass your own if you cannot allocate).  Asynchronous on ``stream``.  Calls that overlap on
    the GPU race on the shared array; the first call on a device should come before any stream capture."""
    import torch
    n = int(pos.shape[0])
    if not (pos.is_cuda and pos.dtype == torch.float64 and pos.is_contiguous() and tuple(pos.shape) == (n, 3)):
        raise DPError("pos must be a contiguous float64 CUDA tensor of shape [n,3]")
    tiles = -(-int(params.nx) // BIN_TILE_X) * -(-int(params.ny) // BIN_TILE_Y)
    if perm is None:
        perm = torch.empty((n,), dtype=torch.int32, device=pos.device)
    if tile_start is None:
        tile_start = torch.empty((tiles + 1,), dtype=torch.int32, device=pos.device)
    for t, m in ((perm, n), (tile_start, tiles + 1)):
        if not (t.is_cuda and t.dtype == torch.int32 and t.is_contiguous() and t.numel() == m):
            raise DPError("perm / tile_start must be contiguous int32 CUDA tensors of n resp. tiles + 1 elements")
    st = stream if stream is not None else torch.cuda.current_stream(pos.device)
    L = load_library()
    rc = L.dp_bin_particles_static(ctypes.byref(params), n, ctypes.c_void_p(pos.data_ptr()), ctypes.c_void_p(perm.data_ptr()),
                                   ctypes.c_void_p(tile_start.data_ptr()), ctypes.c_void_p(st.cuda_stream))
    if rc != 0:
        raise DPError("dp_bin_particles_static failed: %s (%d)" % (L.dp_strerror(rc).decode(), rc))
    return perm, tile_start


STAGE_NAMES = ["bin", "spread", "fft_fwd", "solve", "fft_inv", "interp", "k0", "total"]


class Plan:
    """dp_create / dp_mobility_apply / dp_destroy.  ``prob`` is any object with the fields of ``workloads.Problem``."""

    def __init__(self, prob, max_particles: int, use_torques=None, device: int = 0, fft_backend: int = 0, transfer_fp32: bool = False,
                 dense_planes: bool = False, torque_mode: int = 0, solve_kernel: int = 0):
        self._h = None
        L = load_library()
        if use_torques is None:
            use_torques = bool(getattr(prob, "has_torque", True))
        self.params = dp_params(int(prob.wall_mode), float(prob.Lx), float(prob.Ly), float(prob.H), int(prob.nx), int(prob.ny),
                                int(prob.nz), int(prob.w), float(prob.beta_M), float(prob.beta_D), float(getattr(prob, "a", 1.0)),
                                float(prob.eta), int(max_particles), int(bool(transfer_fp32)), int(device),
                                int(bool(use_torques)), int(fft_backend), int(bool(dense_planes)), int(torque_mode),
                                float(getattr(prob, "slip_0", 0.0)), float(getattr(prob, "slip_H", 0.0)),
                                (ctypes.c_double * 2)(*[float(v) for v in getattr(prob, "uwall_0", (0.0, 0.0))]),
                                (ctypes.c_double * 2)(*[float(v) for v in getattr(prob, "uwall_H", (0.0, 0.0))]),
                                int(solve_kernel))
        h = ctypes.c_void_p()
        rc = L.dp_create(ctypes.byref(self.params), ctypes.byref(h))
        if rc != 0:
            raise DPError("dp_create failed: %s (%d)" % (L.dp_strerror(rc).decode(), rc))
        self._h = h
        self.use_torques = bool(use_torques)
        self.torque_mode = int(torque_mode)
        self.fields = 6 if (use_torques and not torque_mode) else 3
        self.device = device

    # -- lifetime
    def close(self):
        if self._h is not None:
            load_library().dp_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _ck(self, rc, what):
        if rc != 0:
            L = load_library()
            raise DPError("%s failed: %s (%d): %s" % (what, L.dp_strerror(rc).decode(), rc, L.dp_last_error(self._h).decode()))

    # -- the product, device tensors
    def mobility_apply(self, pos, force=None, torque=None, want_omega=None, out_U=None, out_Omega=None, stream=None):
        """(U, Omega) = M (F, tau).  ``pos``, ``force``, ``torque``: float64 CUDA tensors [n,3].  Asynchronous."""
        import torch
        if want_omega is None:
            want_omega = torque is not None
        n = int(pos.shape[0])
        for t in (pos, force, torque):
            if t is not None:
                if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == (n, 3)):
                    raise DPError("arguments must be contiguous float64 CUDA tensors of shape [n,3]")
        U = out_U if out_U is not None else torch.empty((n, 3), dtype=torch.float64, device=pos.device)
        Om = None
        if want_omega:
            Om = out_Omega if out_Omega is not None else torch.empty((n, 3), dtype=torch.float64, device=pos.device)
        st = stream if stream is not None else torch.cuda.current_stream(pos.device)
        ptr = lambda t: None if t is None else ctypes.c_void_p(t.data_ptr())
        rc = load_library().dp_mobility_apply(self._h, n, ptr(pos), ptr(force), ptr(torque), ptr(U), ptr(Om),
                                              ctypes.c_void_p(st.cuda_stream))
        self._ck(rc, "dp_mobility_apply")
        return U, Om

    # -- the product, host arrays (H2D + product + D2H, synchronous)
    def lanczos_sqrt(self, pos, W_force, W_torque=None, tol: float = 1e-3, max_iter: int = 30, stream=None):
        """g = M^{1/2} W by the Lanczos iteration.  CUDA tensors [n,3]; returns (g_U, g_Omega or None, iters, eps list)."""
        import torch
        n = int(pos.shape[0])
        for t in (pos, W_force, W_torque):
            if t is not None:
                assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and tuple(t.shape) == (n, 3)
        gU = torch.empty((n, 3), dtype=torch.float64, device=pos.device)
        gO = torch.empty((n, 3), dtype=torch.float64, device=pos.device) if W_torque is not None else None
        its = ctypes.c_int(0)
        eps = (ctypes.c_double * max(max_iter, 1))()
        ptr = lambda t: ctypes.c_void_p(0 if t is None else t.data_ptr())
        st = torch.cuda.current_stream(pos.device) if stream is None else stream
        rc = load_library().dp_lanczos_sqrt(self._h, n, ptr(pos), ptr(W_force), ptr(W_torque), ptr(gU), ptr(gO), float(tol), int(max_iter),
                                            ctypes.byref(its), eps, ctypes.c_void_p(st.cuda_stream))
        self._ck(rc, "dp_lanczos_sqrt")
        return gU, gO, int(its.value), [float(eps[k]) for k in range(max(int(its.value) - 1, 0))]

    def mobility_apply_host(self, pos, force=None, torque=None, want_omega=None, out_U=None, out_Omega=None):
        if want_omega is None:
            want_omega = torque is not None
        c = lambda a: None if a is None else np.ascontiguousarray(a, dtype=np.float64)
        pos, force, torque = c(pos), c(force), c(torque)
        n = pos.shape[0]
        U = out_U if out_U is not None else np.empty((n, 3))
        Om = (out_Omega if out_Omega is not None else np.empty((n, 3))) if want_omega else None
        ptr = lambda a: None if a is None else a.ctypes.data_as(ctypes.c_void_p)
        rc = load_library().dp_mobility_apply_host(self._h, n, ptr(pos), ptr(force), ptr(torque), ptr(U), ptr(Om))
        self._ck(rc, "dp_mobility_apply_host")
        return U, Om

    def check(self) -> int:
        return int(load_library().dp_check(self._h))

    def set_profiling(self, on: bool):
        self._ck(load_library().dp_set_profiling(self._h, int(on)), "dp_set_profiling")

    def stage_ms(self) -> dict:
        buf = (ctypes.c_float * 8)()
        self._ck(load_library().dp_stage_ms(self._h, buf), "dp_stage_ms")
        return {k: float(buf[i]) for i, k in enumerate(STAGE_NAMES)}

    def fft_pass_ms(self) -> dict:
        buf = (ctypes.c_float * 4)()
        self._ck(load_library().dp_fft_pass_ms(self._h, buf), "dp_fft_pass_ms")
        return {k: float(buf[i]) for i, k in enumerate(("fft_x_fwd", "fft_y_fwd", "fft_y_inv", "fft_x_inv"))}

    def copy_bins(self, n: int):
        """Test hook (dp_copy_bins_to_host): (perm [n], tile_start [tiles+1]) of the last product's own sort, as numpy int32."""
        p = self.params
        tiles = -(-int(p.nx) // BIN_TILE_X) * -(-int(p.ny) // BIN_TILE_Y)
        perm, start = np.empty((n,), dtype=np.int32), np.empty((tiles + 1,), dtype=np.int32)
        self._ck(load_library().dp_copy_bins_to_host(self._h, int(n), perm.ctypes.data_as(ctypes.c_void_p), start.ctypes.data_as(ctypes.c_void_p)),
                 "dp_copy_bins_to_host")
        return perm, start

    def zero_planes(self) -> int:
        return int(load_library().dp_zero_planes(self._h))

    def fft_backend(self) -> str:
        return ["own", "cufft"][int(load_library().dp_fft_backend(self._h))]

    def solve_kernel(self) -> str:
        """Kernel that runs steps 2(z)-6 of a product with three grid fields each way: "pair" (solve_pair.cu) or "tile" (solve.cu)."""
        return ["pair", "tile"][int(load_library().dp_solve_kernel(self._h))]

    def device_bytes(self) -> int:
        return int(load_library().dp_device_bytes(self._h))

    def effective_radius(self, dipole: bool = False) -> float:
        """R_h of the plan's ES kernel (dp_effective_radius): host-side quadrature, no device work."""
        r = float(load_library().dp_effective_radius(self._h, int(bool(dipole))))
        if r < 0:
            raise DPError("dp_effective_radius: invalid request")
        return r

    def copy_plane(self, which: int, field: int, l: int) -> np.ndarray:
        """One xy plane of an internal buffer (test hook): which = 0 real [ny, nx], 1 half spectrum [ny, nx/2+1] (natural layout)."""
        L = load_library()
        p = self.params
        if which == 0:
            out = np.empty((p.ny, p.nx), dtype=np.float64)
        else:
            out = np.empty((p.ny, int(L.dp_complex_row_pitch(self._h))), dtype=np.complex128)
        self._ck(L.dp_copy_plane_to_host(self._h, which, field, l, out.ctypes.data_as(ctypes.c_void_p), out.nbytes), "dp_copy_plane_to_host")
        return out if which == 0 else out[:, : p.nx // 2 + 1]

    def run_stage(self, pos, force, torque, last_stage: int):
        """dp_debug_run_stage without copying anything back (use copy_plane / debug buffers afterwards)."""
        import torch
        ptr = lambda t: None if t is None else ctypes.c_void_p(t.data_ptr())
        st = torch.cuda.current_stream(pos.device)
        self._ck(load_library().dp_debug_run_stage(self._h, int(pos.shape[0]), ptr(pos), ptr(force), ptr(torque), int(last_stage),
                                                    ctypes.c_void_p(st.cuda_stream)), "dp_debug_run_stage")

    # -- test hooks
    def debug_stage(self, pos, force, torque, last_stage: int):
        """Run steps up to ``last_stage`` (1 spread, 2 fwd FFT, 3 solve, 4 inv FFT) and return the stage's buffer as numpy."""
        import torch
        L = load_library()
        n = int(pos.shape[0])
        ptr = lambda t: None if t is None else ctypes.c_void_p(t.data_ptr())
        st = torch.cuda.current_stream(pos.device)
        self._ck(L.dp_debug_run_stage(self._h, n, ptr(pos), ptr(force), ptr(torque), int(last_stage), ctypes.c_void_p(st.cuda_stream)),
                 "dp_debug_run_stage")
        p = self.params
        if last_stage in (1, 4):
            out = np.empty((self.fields, p.nz, p.ny, p.nx), dtype=np.float64)
            self._ck(L.dp_copy_buffer_to_host(self._h, 0, out.ctypes.data_as(ctypes.c_void_p), out.nbytes), "dp_copy_buffer_to_host")
            return out
        pitch = int(L.dp_complex_row_pitch(self._h))
        out = np.empty((self.fields, p.nz, p.ny, pitch), dtype=np.complex128)
        self._ck(L.dp_copy_buffer_to_host(self._h, 1, out.ctypes.data_as(ctypes.c_void_p), out.nbytes), "dp_copy_buffer_to_host")
        return out[..., : p.nx // 2 + 1]
