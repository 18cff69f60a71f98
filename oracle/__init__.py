"""CPU oracle for the doubly-periodic Stokes mobility product (arXiv 2210.01837).

TEST INFRASTRUCTURE — NOT THE PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package.  It shares no code with the CUDA
path and never imports ``paper_2210_01837_b200``.

The arithmetic lives in ``dp_oracle.cpp`` (plain C++, fp64 with long-double dense solves, explicit O(n^2)
DFT sums); this file only builds it, marshals numpy arrays, and strings the paper's eight steps
 together in the paper's order.  The xy transforms (O2, O11) exist in three forms of the SAME sums:
``dft="naive"`` — the explicit O(n^2) sums (the definition); ``dft="fft"`` — the oracle's own plain recursive
mixed-radix FFT in ``dp_oracle.cpp`` (allowed beyond the sizes the naive sums finish, validated
against them in ``tests/test_oracle_basics.py``); ``dft="numpy"`` — ``numpy.fft.rfft2 / irfft2``, kept only as an
independent cross-check of the other two.  Everything else is unchanged by the choice.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import time

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dp_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile dp_oracle.cpp -> liboracle.so (g++ -O2 -fopenmp).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", _SRC, "-o", tmp]
        subprocess.check_call(cmd)
        os.replace(tmp, _LIB)
    return _LIB


class _Params(ctypes.Structure):
    _fields_ = [("wall_mode", ctypes.c_int), ("Lx", ctypes.c_double), ("Ly", ctypes.c_double), ("H", ctypes.c_double),
                ("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int), ("w", ctypes.c_int),
                ("beta_M", ctypes.c_double), ("beta_D", ctypes.c_double), ("eta", ctypes.c_double),
                ("slip_0", ctypes.c_double), ("slip_H", ctypes.c_double), ("uwall_0", ctypes.c_double * 2), ("uwall_H", ctypes.c_double * 2)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        d, i, p = ctypes.c_double, ctypes.c_int, ctypes.c_void_p
        L.or_num_threads.restype = i
        L.or_es_norm.restype = d
        L.or_es_norm.argtypes = [d, d]
        L.or_es_phi.restype = d
        L.or_es_phi.argtypes = [d, d, d, d]
        L.or_es_dphi_cut.restype = d
        L.or_es_dphi_cut.argtypes = [d]
        L.or_es_dphi.restype = d
        L.or_es_dphi.argtypes = [d, d, d, d, d]
        L.or_spread_curl.argtypes = [p, i, p, p, d, p]
        L.or_interp_curl.argtypes = [p, i, p, p, d, p]
        L.or_cheb_nodes.argtypes = [i, d, p]
        L.or_cheb_analysis_matrix.argtypes = [i, p]
        L.or_cheb_synthesis_matrix.argtypes = [i, p]
        L.or_cheb_diff_matrix.argtypes = [i, d, p]
        L.or_cc_weights.argtypes = [i, p]
        L.or_spread.argtypes = [p, i, p, p, d, p]
        L.or_interp.argtypes = [p, i, p, p, d, p]
        L.or_dft_xy_forward.argtypes = [i, i, ctypes.c_long, p, p]
        L.or_dft_xy_inverse.argtypes = [i, i, ctypes.c_long, p, p]
        L.or_fft_xy_forward.argtypes = [i, i, ctypes.c_long, p, p]
        L.or_fft_xy_inverse.argtypes = [i, i, ctypes.c_long, p, p]
        L.or_solve_modes.argtypes = [p, ctypes.c_long, p, p, p, p, p, p]
        L.or_bvp_solve.argtypes = [i, d, d, p, p, p, p]
        L.or_solve.argtypes = [p, p, p, p, p, p]
        _lib = L
    return _lib


def _params(prob) -> _Params:
    """prob: any object with wall_mode, Lx, Ly, H, nx, ny, nz, w, beta_M, beta_D, eta and, optionally, the wall data of App. A /
    eq 27: slip_0, slip_H (partial slip lengths, slit only), uwall_0, uwall_H (uniform wall velocities (x, y))."""
    u0 = tuple(float(v) for v in getattr(prob, "uwall_0", (0.0, 0.0)))
    uH = tuple(float(v) for v in getattr(prob, "uwall_H", (0.0, 0.0)))
    return _Params(int(prob.wall_mode), float(prob.Lx), float(prob.Ly), float(prob.H), int(prob.nx), int(prob.ny),
                   int(prob.nz), int(prob.w), float(prob.beta_M), float(prob.beta_D), float(prob.eta),
                   float(getattr(prob, "slip_0", 0.0)), float(getattr(prob, "slip_H", 0.0)), (ctypes.c_double * 2)(*u0), (ctypes.c_double * 2)(*uH))


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().or_num_threads())


# ---- small pieces (each one formula of the paper) -------------------------------------------------
def es_norm(alpha: float, beta: float) -> float:
    """Z of eq 54."""
    return float(lib().or_es_norm(alpha, beta))


def es_phi(s, alpha: float, beta: float):
    """phi(s; alpha, beta) of eq 54, normalised to unit integral."""
    Z = es_norm(alpha, beta)
    f = lib().or_es_phi
    return np.array([f(float(x), alpha, beta, Z) for x in np.atleast_1d(s)])


def cheb_nodes(nz: int, H: float) -> np.ndarray:
    z = np.empty(nz)
    lib().or_cheb_nodes(nz, H, _ptr(z))
    return z


def cheb_analysis_matrix(nz: int) -> np.ndarray:
    A = np.empty((nz, nz))
    lib().or_cheb_analysis_matrix(nz, _ptr(A))
    return A


def cheb_synthesis_matrix(nz: int) -> np.ndarray:
    S = np.empty((nz, nz))
    lib().or_cheb_synthesis_matrix(nz, _ptr(S))
    return S


def cheb_diff_matrix(nz: int, H: float) -> np.ndarray:
    D = np.empty((nz, nz))
    lib().or_cheb_diff_matrix(nz, H, _ptr(D))
    return D


def cc_weights(nz: int) -> np.ndarray:
    w = np.empty(nz)
    lib().or_cc_weights(nz, _ptr(w))
    return w


def bvp_solve(nz: int, H: float, k: float, r, rhoH=0.0, rho0=0.0) -> np.ndarray:
    """Chebyshev coefficients of y with (d2/dz2 - k^2) y = r, (d/dz + k) y(H) = rhoH, (d/dz - k) y(0) = rho0."""
    r = np.ascontiguousarray(r, dtype=np.complex128)
    assert r.shape == (nz - 2,)
    y = np.empty(nz, dtype=np.complex128)
    a = np.array([rhoH], dtype=np.complex128)
    b = np.array([rho0], dtype=np.complex128)
    lib().or_bvp_solve(nz, H, k, _ptr(r), _ptr(a), _ptr(b), _ptr(y))
    return y


# ---- the eight steps ----------------------------------------------------------------------------------
def spread(prob, pos, val, beta: float) -> np.ndarray:
    """Step 1 (O1): grid[c][l][j][i] = sum_p val[p][c] Delta^W(x_g - r_p)   (eqs 7, 9)."""
    pos, val = _f64(pos), _f64(val)
    P = _params(prob)
    g = np.empty((3, prob.nz, prob.ny, prob.nx))
    lib().or_spread(ctypes.byref(P), pos.shape[0], _ptr(pos), _ptr(val), beta, _ptr(g))
    return g


def interp(prob, pos, grid, beta: float) -> np.ndarray:
    """Step 8 (O12): out[p][c] = sum_g grid[c][g] Delta^W(x_g - r_p) h^2 (H/2) w_l   (eqs 10-11)."""
    pos, grid = _f64(pos), _f64(grid)
    P = _params(prob)
    out = np.empty((pos.shape[0], 3))
    lib().or_interp(ctypes.byref(P), pos.shape[0], _ptr(pos), _ptr(grid), beta, _ptr(out))
    return out


def es_dphi_cut(beta: float) -> float:
    """|s|/alpha beyond which the kernel derivative is truncated to zero (footnote 47)."""
    return float(lib().or_es_dphi_cut(beta))


def es_dphi(s, alpha: float, beta: float, Z: float | None = None, ucut: float | None = None):
    """Truncated derivative of the ES kernel (footnote 47)."""
    Z = es_norm(alpha, beta) if Z is None else Z
    ucut = es_dphi_cut(beta) if ucut is None else ucut
    f = np.vectorize(lambda x: lib().or_es_dphi(float(x), alpha, beta, Z, ucut))
    return f(np.asarray(s, dtype=np.float64))


def spread_curl(prob, pos, torque, beta: float, grid: np.ndarray) -> np.ndarray:
    """Kernel-derivative torque spreading: grid += (1/2) curl_x (tau Delta_D^W)   (eq 7, footnotes 47-48)."""
    pos, torque = _f64(pos), _f64(torque)
    assert grid.shape == (3, prob.nz, prob.ny, prob.nx) and grid.flags.c_contiguous and grid.dtype == np.float64
    P = _params(prob)
    lib().or_spread_curl(ctypes.byref(P), pos.shape[0], _ptr(pos), _ptr(torque), beta, _ptr(grid))
    return grid


def interp_curl(prob, pos, grid, beta: float) -> np.ndarray:
    """Kernel-derivative angular velocity: Omega = (1/2) sum_g u x grad Delta_D^W h^2 (H/2) w_l   (eq 11 by parts)."""
    pos, grid = _f64(pos), _f64(grid)
    P = _params(prob)
    out = np.empty((pos.shape[0], 3))
    lib().or_interp_curl(ctypes.byref(P), pos.shape[0], _ptr(pos), _ptr(grid), beta, _ptr(out))
    return out


def dft_xy_forward(real: np.ndarray, dft: str = "naive") -> np.ndarray:
    """Step 2, xy part (O2): unnormalised forward DFT over the last two axes (j, i) -> half spectrum (ny, nx/2+1)."""
    real = _f64(real)
    ny, nx = real.shape[-2:]
    if dft == "numpy":
        return np.ascontiguousarray(np.fft.rfft2(real, axes=(-2, -1)))
    out = np.empty(real.shape[:-1] + (nx // 2 + 1,), dtype=np.complex128)
    fn = {"naive": lib().or_dft_xy_forward, "fft": lib().or_fft_xy_forward}[dft]
    fn(nx, ny, int(np.prod(real.shape[:-2], dtype=np.int64)), _ptr(real), _ptr(out))
    return out


def dft_xy_inverse(spec: np.ndarray, nx: int, dft: str = "naive") -> np.ndarray:
    """Step 7, xy part (O11): inverse DFT with Hermitian completion and 1/(nx ny)."""
    spec = np.ascontiguousarray(spec, dtype=np.complex128)
    ny = spec.shape[-2]
    if dft == "numpy":
        return np.ascontiguousarray(np.fft.irfft2(spec, s=(ny, nx), axes=(-2, -1)))
    out = np.empty(spec.shape[:-1] + (nx,))
    fn = {"naive": lib().or_dft_xy_inverse, "fft": lib().or_fft_xy_inverse}[dft]
    fn(nx, ny, int(np.prod(spec.shape[:-2], dtype=np.int64)), _ptr(spec), _ptr(out))
    return out


def solve(prob, fh, th=None, want_omega=False, want_coef=False):
    """Steps 2(z)-6 (O3-O10) for every retained (kx, ky): nodal-in-z spectra of f (and t) -> of u (and (1/2) curl u)."""
    fh = np.ascontiguousarray(fh, dtype=np.complex128)
    th = None if th is None else np.ascontiguousarray(th, dtype=np.complex128)
    P = _params(prob)
    uh = np.empty_like(fh)
    wh = np.empty_like(fh) if want_omega else None
    dump = np.empty_like(fh) if want_coef else None
    lib().or_solve(ctypes.byref(P), _ptr(fh), _ptr(th), _ptr(uh), _ptr(wh), _ptr(dump))
    return uh, wh, dump


def solve_modes(prob, ix, iy, fh, th=None, want_omega=False):
    """Steps 2(z)-6 (O3-O10) on a LIST of wavenumbers: column q of ``fh`` / ``th`` ([3, nz, nmodes]) is the nodal-in-z
    spectrum at (kx index ix[q], ky index iy[q] in FFT order).  Same arithmetic as ``solve`` (one body in dp_oracle.cpp)."""
    ix = np.ascontiguousarray(ix, dtype=np.int32)
    iy = np.ascontiguousarray(iy, dtype=np.int32)
    fh = np.ascontiguousarray(fh, dtype=np.complex128)
    th = None if th is None else np.ascontiguousarray(th, dtype=np.complex128)
    assert fh.shape == (3, prob.nz, len(ix)) and len(ix) == len(iy)
    P = _params(prob)
    uh = np.empty_like(fh)
    wh = np.empty_like(fh) if want_omega else None
    lib().or_solve_modes(ctypes.byref(P), len(ix), _ptr(ix), _ptr(iy), _ptr(fh), _ptr(th), _ptr(uh), _ptr(wh))
    return uh, wh


def mobility_apply(prob, pos, force=None, torque=None, want_omega=None, dft="naive", stages=None, timing=None, torque_mode="fourier"):
    """(U, Omega) = M (F, tau): the paper's steps 1-8 in order.

    ``torque_mode``: "fourier" — torques and angular velocities through the curl in Fourier-Chebyshev space (the paper's first
    way); "kernel" — through the derivative of the ES kernel (its second way: three fields each way).

    ``stages`` (dict) receives the intermediate arrays (grid after spread, spectra, ...) when given.
    ``timing`` (dict) receives per-step wall-clock seconds when given.
    Intermediate arrays are released as soon as the next step has consumed them (unless ``stages`` keeps them), so that
    the large configurations fit in host memory.
    """
    if force is None and torque is None:
        raise ValueError("need forces and/or torques")
    if want_omega is None:
        want_omega = torque is not None
    n = np.asarray(pos).shape[0]
    tm = {} if timing is None else timing
    keep = stages is not None
    t0 = time.perf_counter()
    if torque_mode == "kernel":
        f = spread(prob, pos, force if force is not None else np.zeros((n, 3)), prob.beta_M)      # step 1
        if torque is not None:
            spread_curl(prob, pos, torque, prob.beta_D, f)
        tm["spread"] = time.perf_counter() - t0; t0 = time.perf_counter()
        fh = dft_xy_forward(f, dft)                                                                  # step 2 (xy)
        if keep:
            stages.update(f=f)
        del f
        tm["dft_fwd"] = time.perf_counter() - t0; t0 = time.perf_counter()
        uh, _, coef = solve(prob, fh, None, want_omega=False, want_coef=keep)                      # steps 2(z)-6
        if keep:
            stages.update(fh=fh, ucoef=coef)
        del fh, coef
        tm["solve"] = time.perf_counter() - t0; t0 = time.perf_counter()
        u = dft_xy_inverse(uh, prob.nx, dft)                                                         # step 7
        if keep:
            stages.update(uh=uh, u=u)
        del uh
        tm["dft_inv"] = time.perf_counter() - t0; t0 = time.perf_counter()
        U = interp(prob, pos, u, prob.beta_M)                                                        # step 8
        Om = interp_curl(prob, pos, u, prob.beta_D) if want_omega else None
        tm["interp"] = time.perf_counter() - t0
        return U, Om
    assert torque_mode == "fourier"
    f = spread(prob, pos, force if force is not None else np.zeros((n, 3)), prob.beta_M)          # step 1
    t = spread(prob, pos, torque, prob.beta_D) if torque is not None else None
    tm["spread"] = time.perf_counter() - t0; t0 = time.perf_counter()
    fh = dft_xy_forward(f, dft)                                                                      # step 2 (xy)
    th = dft_xy_forward(t, dft) if t is not None else None
    if keep:
        stages.update(f=f, t=t)
    del f, t
    tm["dft_fwd"] = time.perf_counter() - t0; t0 = time.perf_counter()
    uh, wh, coef = solve(prob, fh, th, want_omega=want_omega, want_coef=keep)                     # steps 2(z)-6
    if keep:
        stages.update(fh=fh, th=th, ucoef=coef)
    del fh, th, coef
    tm["solve"] = time.perf_counter() - t0; t0 = time.perf_counter()
    u = dft_xy_inverse(uh, prob.nx, dft)                                                             # step 7
    om = dft_xy_inverse(wh, prob.nx, dft) if want_omega else None
    if keep:
        stages.update(uh=uh, wh=wh)
    del uh, wh
    tm["dft_inv"] = time.perf_counter() - t0; t0 = time.perf_counter()
    U = interp(prob, pos, u, prob.beta_M)                                                            # step 8
    Om = interp(prob, pos, om, prob.beta_D) if want_omega else None
    tm["interp"] = time.perf_counter() - t0
    if keep:
        stages.update(u=u, om=om)
    return U, Om


# ---- Lanczos square root (Sec. V B) ------------------------------------------------------------
def lanczos_sqrt(apply, W, tol: float = 1e-3, max_iter: int = 50):
    """g ~ M^{1/2} W in the Krylov subspace of the symmetric positive definite operator ``apply`` ("A Lanczos iterative
    algorithm [37] can be used to estimate g in the Krylov subspace of M"), step by step:

        v_1 = W/|W|;   for n = 1, 2, ...:   w = M v_n - beta_{n-1} v_{n-1};  alpha_n = w.v_n;  w -= alpha_n v_n;
        beta_n = |w|;  v_{n+1} = w/beta_n;   T_n = tridiag(beta, alpha, beta) (n x n);   g_n = |W| V_n T_n^{1/2} e_1;
        eps_n = |g_n - g_{n-1}| / |g_{n-1}|   (the quantity of Fig. 11);   stop when eps_n < tol.

    T_n^{1/2} through the symmetric eigendecomposition of T_n (library primitive numpy.linalg.eigh).  No reorthogonalisation.
    ``apply`` maps a flat vector to a flat vector.  Returns (g, number of products, [eps_2, eps_3, ...])."""
    W = np.asarray(W, dtype=np.float64).ravel()
    nrm = float(np.linalg.norm(W))
    V = [W / nrm]
    alpha, beta, eps_hist = [], [], []
    g_prev = None
    g = None
    for n in range(1, max_iter + 1):
        w = np.asarray(apply(V[n - 1]), dtype=np.float64).ravel().copy()
        if n > 1:
            w -= beta[n - 2] * V[n - 2]
        a = float(w @ V[n - 1])
        w -= a * V[n - 1]
        b = float(np.linalg.norm(w))
        alpha.append(a); beta.append(b)
        T = np.diag(alpha) + np.diag(beta[:n - 1], 1) + np.diag(beta[:n - 1], -1)
        lam, Q = np.linalg.eigh(T)
        c = Q @ (np.sqrt(np.maximum(lam, 0.0)) * Q[0, :])            # T^{1/2} e_1
        g = nrm * sum(ci * vi for ci, vi in zip(c, V))
        if g_prev is not None:
            eps = float(np.linalg.norm(g - g_prev) / np.linalg.norm(g_prev))
            eps_hist.append(eps)
            if eps < tol:
                return g, n, eps_hist
        g_prev = g
        if b <= 1e-14 * abs(a):                                       # invariant subspace reached: g is exact
            return g, n, eps_hist
        V.append(w / b)
    return g, max_iter, eps_hist
