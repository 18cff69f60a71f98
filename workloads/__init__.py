"""Seeded synthetic inputs for the DP-wall mobility product (shared by oracle tests, GPU tests, bench).

This module holds NONE of the method's arithmetic: it only draws positions, forces and torques and
states the box/grid/kernel parameters of each configuration.  Both the CPU oracle (``oracle/``) and the
CUDA path (``paper_2210_01837_b200/``) consume these arrays; neither imports the other.

The recipes stand in for the paper's workloads (PAPER.md:492, 505 — Fig. 9: particles uniform in the
plane at area fraction 0.4 with a near-wall height distribution; PAPER.md:418 — validation boxes), which
are not in the container; they follow BASELINE.json ``configs`` as read in SURVEY.md §8(d) (G8, G9, G17).

Random numbers: ``numpy.random.Generator(PCG64(seed + i))`` with one stream per array:
i=0 -> x,y ; i=1 -> z ; i=2 -> forces ; i=3 -> torques.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

BOTTOM_WALL = 0
SLIT = 1

# ES parameters from the paper's tables: beta/w for w = 6
BETA_OVER_W_M_ONLY_W6 = 1.714      # Table II, monopole only
BETA_OVER_W_M_W6 = 1.327           # Table I, monopole (with dipole)
BETA_OVER_W_D_W6 = 2.216           # Table I, dipole
BETA_OVER_W_M_ONLY_W4 = 1.785      # Table II, w = 4


@dataclasses.dataclass(frozen=True)
class Problem:
    """Box, grid and kernel parameters (plain numbers only)."""
    name: str
    wall_mode: int          # BOTTOM_WALL or SLIT
    Lx: float               # FULL period in x
    Ly: float
    H: float                # top of the z grid (open for BOTTOM_WALL, wall for SLIT)
    nx: int
    ny: int
    nz: int
    w: int                  # ES support in cells (paper's m)
    beta_M: float           # ES beta (not beta/w)
    beta_D: float
    eta: float = 1.0
    a: float = 1.0          # nominal radius (informational)
    has_torque: bool = True     # torques in, Omega out
    seed: int = 0
    n: int = 0
    # wall data of Appendix A / eq 27: partial slip lengths (slit only) and uniform wall velocities (x, y)
    slip_0: float = 0.0
    slip_H: float = 0.0
    uwall_0: tuple = (0.0, 0.0)
    uwall_H: tuple = (0.0, 0.0)

    @property
    def h(self) -> float:
        return self.Lx / self.nx

    @property
    def alpha(self) -> float:
        return 0.5 * self.w * self.h


def smooth_at_least(n: int) -> int:
    """Smallest integer >= n of the form 2^a 3^b 5^c 7^d that is even."""
    m = max(2, int(n))
    while True:
        r = m
        for p in (2, 3, 5, 7):
            while r % p == 0:
                r //= p
        if r == 1 and m % 2 == 0:
            return m
        m += 1


def _rng(seed: int, i: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed + i))


def _xy(seed: int, n: int, Lx: float, Ly: float) -> np.ndarray:
    g = _rng(seed, 0)
    return np.stack([g.uniform(0.0, Lx, n), g.uniform(0.0, Ly, n)], axis=1)


def _pack(xy: np.ndarray, z: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(np.concatenate([xy, z[:, None]], axis=1), dtype=np.float64)


def _normal(seed: int, i: int, n: int, sigma: float = 1.0) -> np.ndarray:
    return np.ascontiguousarray(_rng(seed, i).normal(0.0, sigma, (n, 3)), dtype=np.float64)


def _roller_drive(seed: int, n: int):
    """Forces -z (unit gravity) + N(0, 0.1^2) noise; torques +y of unit magnitude (config 3 recipe)."""
    F = _normal(seed, 2, n, 0.1)
    F[:, 2] -= 1.0
    T = np.zeros((n, 3), dtype=np.float64)
    T[:, 1] = 1.0
    return F, T


def monolayer_L(n: int, phi: float = 0.4, a: float = 1.0) -> float:
    return math.sqrt(n * math.pi * a * a / phi)


def random_bw(n=128, L=32.0, nxy=48, nz=32, H=8.0, zlo=1.5, zhi=5.0, seed=1001, name="cfg1"):
    """Config 1: bottom wall, forces only, uniform positions."""
    prob = Problem(name, BOTTOM_WALL, L, L, H, nxy, nxy, nz, 6, 6 * BETA_OVER_W_M_ONLY_W6, 0.0,
                   has_torque=False, seed=seed, n=n)
    pos = _pack(_xy(seed, n, L, L), _rng(seed, 1).uniform(zlo, zhi, n))
    return prob, pos, _normal(seed, 2, n), None


def random_slit(n=4096, L=128.0, nxy=192, nz=48, H=8.0, margin=1.5, seed=1002, name="cfg2"):
    """Config 2: slit channel, forces and torques N(0,1), z uniform in [margin, H-margin]."""
    prob = Problem(name, SLIT, L, L, H, nxy, nxy, nz, 6, 6 * BETA_OVER_W_M_W6, 6 * BETA_OVER_W_D_W6,
                   seed=seed, n=n)
    pos = _pack(_xy(seed, n, L, L), _rng(seed, 1).uniform(margin, H - margin, n))
    return prob, pos, _normal(seed, 2, n), _normal(seed, 3, n)


def _xy_jittered_lattice(seed: int, n: int, L: float, a: float = 1.0) -> np.ndarray:
    """Non-overlapping in-plane positions at the same area fraction: a square lattice of sqrt(n) x sqrt(n) sites of spacing d = L / sqrt(n)
    (d = 2.80 a at area fraction 0.4), every site displaced uniformly by up to (d - 2a)/2 in x and in y, so that two centres are never closer
    than 2a in the plane — the hard-disk constraint of the paper's equilibrated tile, which uniform draws violate (density
    spikes).  Site order is shuffled so that particle index carries no spatial order, as in the uniform recipe."""
    m = int(round(math.sqrt(n)))
    if m * m != n:
        raise ValueError("the jittered lattice needs a square number of particles")
    d = L / m
    if d < 2.0 * a:
        raise ValueError("area fraction too high for a non-overlapping square lattice")
    g = _rng(seed, 0)
    ij = g.permutation(n)
    jit = g.uniform(-0.5 * (d - 2.0 * a), 0.5 * (d - 2.0 * a), (n, 2))
    xy = np.stack([(ij % m + 0.5) * d, (ij // m + 0.5) * d], axis=1) + jit
    return xy


def monolayer_bw(n=65536, nz=32, H=13.0, seed=1003, name="cfg3", zclip=11.0, xy="uniform"):
    """Configs 3, 5: sedimented microroller monolayer above one wall at area fraction 0.4.  xy = "uniform" (BASELINE.json's recipe) or
    "jittered": the non-overlapping jittered-lattice stand-in of SURVEY.md §8(d), same box, grid, heights and drives."""
    L = monolayer_L(n)
    nxy = smooth_at_least(math.ceil(1.5 * L))
    prob = Problem(name, BOTTOM_WALL, L, L, H, nxy, nxy, nz, 6, 6 * BETA_OVER_W_M_W6,
                   6 * BETA_OVER_W_D_W6, seed=seed, n=n)
    z = np.minimum(1.0 + _rng(seed, 1).exponential(0.5, n), zclip)
    F, T = _roller_drive(seed, n)
    if xy not in ("uniform", "jittered"):
        raise ValueError("xy must be 'uniform' or 'jittered'")
    pxy = _xy(seed, n, L, L) if xy == "uniform" else _xy_jittered_lattice(seed, n, L)
    return prob, _pack(pxy, z), F, T


def monolayer_slit(n=262144, nz=48, H=6.0, margin=1.2, seed=1004, name="cfg4"):
    """Config 4: microrollers in a slit channel of height H at area fraction 0.4."""
    L = monolayer_L(n)
    nxy = smooth_at_least(math.ceil(1.5 * L))
    prob = Problem(name, SLIT, L, L, H, nxy, nxy, nz, 6, 6 * BETA_OVER_W_M_W6, 6 * BETA_OVER_W_D_W6,
                   seed=seed, n=n)
    z = _rng(seed, 1).uniform(margin, H - margin, n)
    F, T = _roller_drive(seed, n)
    return prob, _pack(_xy(seed, n, L, L), z), F, T


def paper_fig9(replicas: int = 18, dipole: bool = False, seed: int = 1009, name: str | None = None):
    """Stand-in for the paper's own performance workload (Fig. 9 and Table III): a tile of 2048 particles of
    size L = 128.8 R_h, replicated ``replicas`` x ``replicas`` times in the plane (18 x 18 = 663,552 particles is its largest case),
    area fraction 0.4, two layers of heights above the wall ("bimodal", the inset of Fig. 9), H = 9.1 R_h (M) / 9.2 R_h (M & D).
    Grid and kernels are Table III's: M (forces only): Nz = 19, Nxy = 150 per tile, m = 4, beta/m = 1.87;  M & D: Nz = 26,
    Nxy = 216 per tile, m = 6, beta_M/m = 1.38, beta_D/m = 2.3.  R_h = 1.  The tile of ref. [22] itself is not in the container:
    positions are drawn uniformly (not replicated), heights 1 + Exp(0.3) for two thirds of the particles and N(3.2, 0.3^2) for
    the rest, clipped to [0.8, H - alpha]."""
    n = 2048 * replicas * replicas
    L = 128.8 * replicas
    if dipole:
        H, nz, nxy, w, bM, bD = 9.2, 26, 216 * replicas, 6, 6 * 1.38, 6 * 2.3
    else:
        H, nz, nxy, w, bM, bD = 9.1, 19, 150 * replicas, 4, 4 * 1.87, 0.0
    prob = Problem(name or ("fig9-%s-%dx%d" % ("MD" if dipole else "M", replicas, replicas)), BOTTOM_WALL, L, L, H, nxy, nxy, nz, w, bM, bD,
                   has_torque=dipole, seed=seed, n=n)
    g = _rng(seed, 1)
    low = 1.0 + g.exponential(0.3, n)
    high = g.normal(3.2, 0.3, n)
    z = np.where(g.uniform(0.0, 1.0, n) < 2.0 / 3.0, low, high)
    z = np.clip(z, 0.8, H - prob.alpha)
    F, T = _roller_drive(seed, n)
    return prob, _pack(_xy(seed, n, L, L), z), F, (T if dipole else None)


def config(i: int):
    """BASELINE.json ``configs[i-1]`` (1-based, as SURVEY.md numbers them)."""
    if i == 1:
        return random_bw()
    if i == 2:
        return random_slit()
    if i == 3:
        return monolayer_bw()
    if i == 4:
        return monolayer_slit()
    if i == 5:
        return monolayer_bw(n=1048576, seed=1005, name="cfg5")
    raise ValueError("config index must be 1..5")


def describe(prob: Problem) -> dict:
    d = dataclasses.asdict(prob)
    d["h"] = prob.h
    return d
