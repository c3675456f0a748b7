"""Pins for the oracle's full Ewald sum (oracle/ewald_ref.c) against things the paper and the
mathematics fix independently of it: the rock-salt Madelung constant, alpha-independence,
finite differences of the energy, and a brute-force periodic image sum (+ dipole term).

These establish signs, 4 pi / V prefactors and the Gaussian-unit convention of Eqs. (2.8),
(2.10), (2.11); test_oracle_rbe.py then ties Eq. (2.12) to Eq. (2.11).
"""
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _golden_value(fname, key):
    with open(os.path.join(GOLDEN, fname)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line.startswith(key + " "):
                return float(line.split()[1])
    raise KeyError(key)


def _rocksalt():
    """8-ion NaCl cell, lattice constant a = 2 (nearest-neighbour distance 1)."""
    r, q = [], []
    for i in range(2):
        for j in range(2):
            for k in range(2):
                r.append([i, j, k])
                q.append((-1.0) ** (i + j + k))
    return np.array(r, dtype=np.float64), np.array(q), 2.0


def _random_neutral(n, L, seed, min_sep=0.5):
    rng = np.random.default_rng(seed)
    while True:
        r = rng.random((n, 3)) * L
        d = r[:, None, :] - r[None, :, :]
        d -= L * np.round(d / L)
        dist = np.sqrt((d ** 2).sum(-1)) + np.eye(n) * 10
        if dist.min() > min_sep:
            break
    q = rng.uniform(0.5, 1.5, n) * np.where(np.arange(n) % 2 == 0, 1.0, -1.0)
    q -= q.mean()
    return r, q


@pytest.mark.parametrize("alpha", [1.0, 2.0, 4.0])
def test_madelung_constant_nacl(alpha):
    """U_cell = -4 M for the 8-ion cell with r0 = 1; M = 1.7475645946 (BASELINE.json north_star:
    'reproduces the Madelung constant 1.747565 to 1e-6').  alpha-independence of the total is a
    second invariant: only the split between the three terms of Eq. (2.8) may move."""
    M_ref = _golden_value("madelung_nacl.txt", "madelung_nacl")
    r, q, L = _rocksalt()
    U, Fs, Fl = oracle.ewald_full(r, q, L, alpha, nreal=5, mmax=12)
    M = -U.sum() / 4.0
    assert abs(M - M_ref) < 1e-10, (alpha, M)
    # by symmetry every ion sits at an inversion centre: no net force
    assert np.abs(Fs + Fl).max() < 1e-12


def test_split_moves_with_alpha_total_does_not():
    r, q = _random_neutral(6, 3.0, 11)
    tot, parts = [], []
    for alpha in (0.8, 1.5, 3.0):
        U, Fs, Fl = oracle.ewald_full(r, q, 3.0, alpha, nreal=5, mmax=14)
        tot.append((U.sum(), Fs + Fl))
        parts.append(U[1])
    assert abs(parts[0] - parts[2]) > 1e-3  # the split really changes
    for u, f in tot[1:]:
        assert abs(u - tot[0][0]) < 1e-10
        assert np.abs(f - tot[0][1]).max() < 1e-10


def test_forces_are_minus_gradient_of_energy():
    """Eq. (2.10) = -grad U_real and Eq. (2.11) = -grad U_k, term by term (signs, prefactors)."""
    L, alpha, h = 3.0, 1.2, 1e-5
    r, q = _random_neutral(5, L, 3)
    U, Fs, Fl = oracle.ewald_full(r, q, L, alpha, nreal=4, mmax=10)
    for i in range(5):
        for d in range(3):
            rp, rm = r.copy(), r.copy()
            rp[i, d] += h
            rm[i, d] -= h
            Up, _, _ = oracle.ewald_full(rp, q, L, alpha, nreal=4, mmax=10)
            Um, _, _ = oracle.ewald_full(rm, q, L, alpha, nreal=4, mmax=10)
            g = (Up - Um) / (2 * h)
            assert abs(-g[0] - Fs[i, d]) < 2e-8, ("short", i, d)
            assert abs(-g[1] - Fl[i, d]) < 2e-8, ("long", i, d)
            assert abs(g[2]) < 1e-12  # self term does not depend on positions


@pytest.mark.parametrize("n,seed", [(2, 5), (4, 6), (8, 7)])
def test_ewald_matches_brute_force_image_sum(n, seed):
    """Total Ewald force (Eq. 2.10 + 2.11) against the literal image sum of Eq. (2.5) over a
    sphere of cells.  Spherical summation gives the vacuum-boundary result, Ewald the tin-foil
    one; they differ by the dipole term (2 pi/3V)|M|^2, i.e. F_i^sphere = F_i^Ewald -
    (4 pi/3V) q_i M with M = sum_j q_j r_j.  Without that term the mismatch is O(1)."""
    L, R = 3.0, 40
    r, q = _random_neutral(n, L, seed)
    U, Fs, Fl = oracle.ewald_full(r, q, L, 1.0, nreal=4, mmax=9)
    Ud, Fd = oracle.direct_image_sum(r, q, L, R)
    Mdip = (q[:, None] * r).sum(0)
    V = L ** 3
    F_ew = Fs + Fl
    F_direct_tinfoil = Fd + 4 * np.pi / (3 * V) * q[:, None] * Mdip[None, :]
    rel = np.linalg.norm(F_direct_tinfoil - F_ew) / np.linalg.norm(F_ew)
    assert rel < 1e-6, rel
    # and the dipole term is not a no-op for this configuration
    rel_without = np.linalg.norm(Fd - F_ew) / np.linalg.norm(F_ew)
    assert rel_without > 100 * rel
    # energies: U_sphere = U_Ewald + (2 pi/3V)|M|^2
    assert abs(Ud - (U.sum() + 2 * np.pi / (3 * V) * (Mdip ** 2).sum())) < 5e-5 * abs(Ud)
