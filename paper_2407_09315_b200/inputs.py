"""Seeded synthetic inputs for the RBE k-space path (numpy only).

This module is the ONE piece shared by the CUDA path's callers and the oracle's tests: it
produces the atom records ``float32 [N,4] = {x, y, z, q}`` and the integer wavevector sets
``int32 [P,3]`` that both sides receive identically.  It holds none of the arithmetic of
Eq. (2.9) / Eq. (2.12); it imports neither ``oracle`` nor the CUDA binding.

The inputs are synthetic stand-ins for the paper's SPC/E water and primitive-electrolyte
systems, whose input files are not available: shapes, densities and
charges follow BASELINE.json ``configs``; the recipe is stated in DESIGN.md section 3.

k-sampling (Algorithm 1 step 1): the paper draws k ~ exp(-k^2/4alpha)/Q,
k != 0, by Metropolis on the CPU with unstated proposal/burn-in.  Here (reading Q2)
the same distribution is sampled exactly and iid: with k = 2 pi m / L the pmf factorises,
p(m) ~ prod_d exp(-pi^2 m_d^2 / (alpha L^2)), so each component is drawn from the 1-D
discrete Gaussian by inverse CDF and the triple (0,0,0) is rejected.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

ALPHA = 0.09  # A^-2, every BASELINE.json config
DENSITY = 0.1  # atoms / A^3

Q_O = np.float32(-0.8476)
Q_H = np.float32(0.4238)
# H offsets in the molecular frame for |OH| = 1.0 A and H-O-H = 109.47 deg
_H_LOCAL = np.array([[0.816490, 0.577359, 0.0], [-0.816490, 0.577359, 0.0]])


@dataclass(frozen=True)
class Config:
    name: str
    N: int
    L: float
    P: int
    seed: int
    kind: str  # "water", "water+nacl", "ions"
    n_water: int = 0
    n_ion_pairs: int = 0
    alpha: float = ALPHA


def ion_box(N: int) -> float:
    return float((N / DENSITY) ** (1.0 / 3.0))


# BASELINE.json configs 1-4 (index 0-3) and the random-ion sweep (config 5)
CONFIGS = {
    "water_3k": Config("water_3k", 3_000, 31.04, 100, 1, "water", n_water=1_000),
    "water_96k": Config("water_96k", 96_000, 98.65, 100, 2, "water", n_water=32_000),
    # DESIGN.md reading Q13: 332 731 waters + 903 Na+ + 903 Cl- = 999 999 atoms
    "water_nacl_1m": Config("water_nacl_1m", 999_999, 215.443, 200, 3, "water+nacl",
                            n_water=332_731, n_ion_pairs=903),
    "water_10m": Config("water_10m", 9_999_999, 464.159, 200, 4, "water", n_water=3_333_333),
}


def ions_config(N: int, P: int = 200) -> Config:
    """Config 5: neutral +-1 e ions, uniform, 0.1 atoms/A^3, seed 5."""
    assert N % 2 == 0
    return Config(f"ions_{N}_P{P}", N, ion_box(N), P, 5, "ions", n_ion_pairs=N // 2)


def _rotation_from_quaternion(qn: np.ndarray) -> np.ndarray:
    """Rotation matrices [n,3,3] from unit quaternions [n,4] = (w, x, y, z)."""
    w, x, y, z = qn[:, 0], qn[:, 1], qn[:, 2], qn[:, 3]
    R = np.empty((qn.shape[0], 3, 3), dtype=np.float64)
    R[:, 0, 0] = 1 - 2 * (y * y + z * z)
    R[:, 0, 1] = 2 * (x * y - z * w)
    R[:, 0, 2] = 2 * (x * z + y * w)
    R[:, 1, 0] = 2 * (x * y + z * w)
    R[:, 1, 1] = 1 - 2 * (x * x + z * z)
    R[:, 1, 2] = 2 * (y * z - x * w)
    R[:, 2, 0] = 2 * (x * z - y * w)
    R[:, 2, 1] = 2 * (y * z + x * w)
    R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def _waters(rng: np.random.Generator, n: int, L: float) -> np.ndarray:
    """n rigid SPC/E-like waters, atom order O,H,H; H atoms are NOT wrapped into the box."""
    out = np.empty((n, 3, 4), dtype=np.float64)
    O = rng.random((n, 3)) * L
    quat = rng.standard_normal((n, 4))
    quat /= np.linalg.norm(quat, axis=1, keepdims=True)
    R = _rotation_from_quaternion(quat)
    out[:, 0, :3] = O
    out[:, 1, :3] = O + np.einsum("nij,j->ni", R, _H_LOCAL[0])
    out[:, 2, :3] = O + np.einsum("nij,j->ni", R, _H_LOCAL[1])
    out[:, 0, 3] = float(Q_O)
    out[:, 1, 3] = float(Q_H)
    out[:, 2, 3] = float(Q_H)
    return out.reshape(3 * n, 4)


def _ions(rng: np.random.Generator, n_pairs: int, L: float) -> np.ndarray:
    """2*n_pairs point charges +1, -1 alternating, uniform in the box."""
    out = np.empty((2 * n_pairs, 4), dtype=np.float64)
    out[:, :3] = rng.random((2 * n_pairs, 3)) * L
    out[0::2, 3] = 1.0
    out[1::2, 3] = -1.0
    return out


def make_atoms(cfg: Config) -> np.ndarray:
    """float32 [N,4] = {x,y,z,q}: drawn in fp64 with PCG64(seed), cast to fp32 at the end."""
    rng = np.random.default_rng(cfg.seed)
    parts = []
    if cfg.n_water:
        parts.append(_waters(rng, cfg.n_water, cfg.L))
    if cfg.n_ion_pairs:
        parts.append(_ions(rng, cfg.n_ion_pairs, cfg.L))
    a = np.concatenate(parts, axis=0)
    assert a.shape[0] == cfg.N, (a.shape, cfg.N)
    return np.ascontiguousarray(a.astype(np.float32))


MASS_NA, MASS_CL = 22.98977, 35.453  # amu


def rocksalt(ncells: int, a: float = 5.64, seed: int = 7, jitter: float = 0.05, v_rms: float = 0.0):
    """A perturbed rock-salt (NaCl) crystal for the NVE loop: ncells^3 conventional cells of
    side a [A] (8 ions each: Na+ on the fcc sites, Cl- shifted by a/2 along x), every ion displaced by a normal
    deviate of standard deviation `jitter` [A], velocities normal with per-component deviation v_rms / sqrt(m)
    [A / tau] minus the centre-of-mass drift.  Returns (x fp64 [N,3], v fp64 [N,3], q fp32 [N], mass fp64 [N], L)."""
    rng = np.random.default_rng(seed)
    fcc = np.array([[0.0, 0.0, 0.0], [0.0, 0.5, 0.5], [0.5, 0.0, 0.5], [0.5, 0.5, 0.0]])
    cells = np.stack(np.meshgrid(*[np.arange(ncells)] * 3, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    na = (cells + fcc[None]).reshape(-1, 3)
    cl = na + np.array([0.5, 0.0, 0.0])
    x = np.concatenate([na, cl]) * a
    n = x.shape[0]
    q = np.concatenate([np.ones(n // 2), -np.ones(n // 2)]).astype(np.float32)
    mass = np.concatenate([np.full(n // 2, MASS_NA), np.full(n // 2, MASS_CL)])
    x = x + jitter * rng.standard_normal((n, 3))
    v = v_rms * rng.standard_normal((n, 3)) / np.sqrt(mass)[:, None]
    v -= (mass[:, None] * v).sum(0) / mass.sum()
    return x, v, q, mass, float(ncells * a)


def plasma(ncells: int, a: float = 4.0, seed: int = 7, jitter: float = 0.05, v_rms: float = 0.0):
    """A one-component plasma for LONG NVE runs: ncells^3 body-centred cubic cells of side a [A]
    (2 ions each), every ion with charge +1 e and the mass of Na; the k = 0 term is absent from Eq. (2.8), i.e. a
    uniform neutralising background is implied (reading Q8), and it exerts no force.  Like charges repel, so -- unlike
    the rock-salt crystal -- nothing collapses on a path without a repulsive core, and the energy error of a long run
    measures the integrator and the random batch only.  Displacements, velocities and return values as rocksalt()."""
    rng = np.random.default_rng(seed)
    cells = np.stack(np.meshgrid(*[np.arange(ncells)] * 3, indexing="ij"), axis=-1).reshape(-1, 1, 3)
    x = (cells + np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.5]])[None]).reshape(-1, 3) * a
    n = x.shape[0]
    q = np.ones(n, dtype=np.float32)
    mass = np.full(n, MASS_NA)
    x = x + jitter * rng.standard_normal((n, 3))
    v = v_rms * rng.standard_normal((n, 3)) / np.sqrt(mass)[:, None]
    v -= (mass[:, None] * v).sum(0) / mass.sum()
    return x, v, q, mass, float(ncells * a)


def pmf_1d(L: float, alpha: float):
    """(support m = -M..M, probabilities) of the 1-D discrete Gaussian exp(-pi^2 m^2/(alpha L^2))."""
    c = np.pi ** 2 / (alpha * L * L)
    M = int(np.ceil(np.sqrt(745.0 / c))) + 1  # exp(-745) underflows in fp64
    ms = np.arange(-M, M + 1, dtype=np.int64)
    p = np.exp(-c * ms.astype(np.float64) ** 2)
    return ms, p / p.sum()


def sample_kset(L: float, alpha: float, P: int, seed: int, step: int = 0) -> np.ndarray:
    """int32 [P,3]: P iid draws of m != 0 with probability ~ exp(-|2 pi m/L|^2 / 4 alpha).

    With replacement; duplicates are kept (each sample carries weight S/P); k and -k are both
    in the support.  Generator: PCG64 seeded with [seed, step].
    """
    rng = np.random.default_rng([seed, step])
    ms, p = pmf_1d(L, alpha)
    cdf = np.cumsum(p)
    cdf[-1] = 1.0
    out = np.empty((P, 3), dtype=np.int32)
    filled = 0
    p_accept = 1.0 - float(p[ms == 0][0]) ** 3
    while filled < P:
        n = int(min(4_000_000, max(16, (P - filled) / max(p_accept, 1e-12) * 1.1)))
        u = rng.random((n, 3))
        idx = np.minimum(np.searchsorted(cdf, u, side="right"), len(ms) - 1)
        cand = ms[idx]
        cand = cand[np.any(cand != 0, axis=1)][: P - filled]
        out[filled:filled + cand.shape[0]] = cand
        filled += cand.shape[0]
    return out


def full_kgrid(mmax: int) -> np.ndarray:
    """Every m in Z^3 with |m_d| <= mmax, m != 0 (for the deterministic-Ewald mode)."""
    r = np.arange(-mmax, mmax + 1, dtype=np.int32)
    g = np.stack(np.meshgrid(r, r, r, indexing="ij"), axis=-1).reshape(-1, 3)
    return np.ascontiguousarray(g[np.any(g != 0, axis=1)])


def shard_bounds(N: int, world_size: int, rank: int, align: int = 1):
    """Contiguous, balanced atom range [lo, hi) of `rank` (multi-GPU sharding)."""
    lo = (N * rank) // world_size
    hi = (N * (rank + 1)) // world_size
    if align > 1:
        lo = min(N, (lo + align - 1) // align * align) if rank > 0 else 0
        hi = min(N, (hi + align - 1) // align * align) if rank < world_size - 1 else N
    return lo, hi
