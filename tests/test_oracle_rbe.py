"""Pins for the RBE oracle (oracle/rbe_oracle.c): Eq. (2.9), Eq. (2.12), the energy estimate
and the normaliser S, against closed forms, invariants, brute force on tiny inputs and the
deterministic Ewald k-space force (itself pinned in test_oracle_ewald.py).

A plausible mistake anywhere -- a dropped 4 pi / V, Q/P, 1/k^2; a wrong sign; Re/Im swapped;
k instead of k/k^2; a transposed index -- fails at least one test here.
"""
import numpy as np
import pytest

import oracle
from paper_2407_09315_b200 import inputs


def _atoms(n, L, seed, neutral=True):
    """fp32-exact random atoms (positions on a 2^-12 grid so that fp64 copies are identical)."""
    rng = np.random.default_rng(seed)
    r = np.round(rng.random((n, 3)) * L * 4096) / 4096
    q = np.round(rng.uniform(-1, 1, n) * 1024) / 1024
    if neutral and n > 1:
        q[-1] = -q[:-1].sum()
    return np.concatenate([r, q[:, None]], axis=1).astype(np.float32)


def _kvec(m, L):
    return 2 * np.pi * np.asarray(m, dtype=np.float64) / L


# --------------------------------------------------------------------------- S
@pytest.mark.parametrize("L,alpha", [(31.04, 0.09), (6.0, 0.5), (3.0, 1.0), (98.65, 0.09)])
def test_S_three_routes(L, alpha):
    """S = H^3 - 1 equals (i) the literal 3-D grid sum and (ii) the Poisson-resummed form
    H = L sqrt(alpha/pi) (1 + 2 sum_n exp(-alpha L^2 n^2))."""
    s = oracle.S(L, alpha)
    c = np.pi ** 2 / (alpha * L * L)
    mmax = int(np.ceil(np.sqrt(40.0 / c)))
    if mmax <= 40:
        assert abs(oracle.S_grid(L, alpha, mmax) - s) < 1e-11 * max(1.0, s)
    n = np.arange(1, 200, dtype=np.float64)
    H = L * np.sqrt(alpha / np.pi) * (1 + 2 * np.exp(-alpha * L * L * n * n).sum())
    assert abs((H ** 3 - 1) - s) < 1e-11 * max(1.0, s)


# ----------------------------------------------------------- rho, closed forms
def test_rho_single_atom_and_axes():
    """One charge q at r: rho(k) = q exp(i k.r).  Distinguishes x/y/z and Re/Im."""
    L = 8.0
    a = np.array([[1.0, 2.5, 0.75, -0.5]], dtype=np.float32)
    m = np.array([[1, 0, 0], [0, 1, 0], [0, 0, 1], [2, -1, 3]], dtype=np.int32)
    rho = oracle.rho(a, L, m)
    for l in range(4):
        ph = 2 * np.pi * (m[l] * a[0, :3].astype(np.float64)).sum() / L
        assert abs(rho[l, 0] - (-0.5) * np.cos(ph)) < 1e-14
        assert abs(rho[l, 1] - (-0.5) * np.sin(ph)) < 1e-14


def test_single_atom_has_no_force():
    a = _atoms(1, 5.0, 0, neutral=False)
    m = inputs.sample_kset(5.0, 0.5, 16, 1)
    S = oracle.S(5.0, 0.5)
    F = oracle.force(a, 5.0, m, S, oracle.rho(a, 5.0, m))
    assert np.abs(F).max() < 1e-15


def test_two_charges_one_k_closed_form():
    """F_1 = -(4 pi S q1 q2 / (V P)) (k/k^2) sin(k.(r2 - r1)), F_2 = -F_1  (from Eq. 2.12 with
    rho = q1 e^{ik.r1} + q2 e^{ik.r2}); like charges at a quarter wavelength repel."""
    L, alpha = 8.0, 0.4
    S = oracle.S(L, alpha)
    m = np.array([[1, 0, 0]], dtype=np.int32)
    a = np.array([[1.0, 3.0, 3.0, 0.5], [3.0, 3.0, 3.0, 0.25]], dtype=np.float32)  # dx = L/4
    F = oracle.force(a, L, m, S, oracle.rho(a, L, m))
    k = _kvec(m[0], L)
    expect = -(4 * np.pi * S * 0.5 * 0.25 / (L ** 3 * 1)) * k / (k @ k) * np.sin(k @ np.array([2.0, 0, 0]))
    assert np.abs(F[0] - expect).max() < 1e-15
    assert np.abs(F[1] + expect).max() < 1e-15
    assert F[0, 0] < 0 < F[1, 0]  # atom 1 (left) pushed left, atom 2 pushed right: repulsion
    assert abs(F[0, 1]) + abs(F[0, 2]) < 1e-16


def test_pair_form_brute_force():
    """Eq. (2.12) expanded into pairs: F_i = (4 pi S q_i/(V P)) sum_l (k_l/k_l^2) sum_j q_j
    sin(k_l.(r_i - r_j)) -- pure numpy, no structure factor."""
    L, alpha, P = 7.0, 0.3, 9
    a = _atoms(7, L, 21)
    m = inputs.sample_kset(L, alpha, P, 4)
    S = oracle.S(L, alpha)
    F = oracle.force(a, L, m, S, oracle.rho(a, L, m))
    r, q = a[:, :3].astype(np.float64), a[:, 3].astype(np.float64)
    ref = np.zeros((7, 3))
    for i in range(7):
        for l in range(P):
            k = _kvec(m[l], L)
            s = sum(q[j] * np.sin(k @ (r[i] - r[j])) for j in range(7))
            ref[i] += 4 * np.pi * S * q[i] / (L ** 3 * P) * k / (k @ k) * s
    assert np.abs(F - ref).max() < 1e-14


# ---------------------------------------------------------------- invariants
@pytest.fixture(scope="module")
def system():
    L, alpha, P = 8.0, 0.35, 40
    a = _atoms(50, L, 5)
    m = inputs.sample_kset(L, alpha, P, 9)
    S = oracle.S(L, alpha)
    rho = oracle.rho(a, L, m)
    F = oracle.force(a, L, m, S, rho)
    return L, alpha, P, a, m, S, rho, F


def test_momentum_conservation(system):
    """sum_i F_i = 0 for EVERY k-set: sum_i q_i Im(e^{-ik.r_i} rho) = Im |rho|^2 = 0."""
    L, alpha, P, a, m, S, rho, F = system
    assert np.abs(F.sum(0)).max() < 1e-13 * np.abs(F).sum()
    for l in range(0, P, 7):  # and per single k
        Fl = oracle.force(a, L, m[l:l + 1], S, rho[l:l + 1])
        assert np.abs(Fl.sum(0)).max() < 1e-13 * np.abs(Fl).sum()


def test_sign_flip_of_m_leaves_force(system):
    L, alpha, P, a, m, S, rho, F = system
    m2 = m.copy()
    m2[::2] *= -1
    rho2 = oracle.rho(a, L, m2)
    assert np.abs(rho2[::2, 0] - rho[::2, 0]).max() < 1e-12  # rho(-k) = conj rho(k)
    assert np.abs(rho2[::2, 1] + rho[::2, 1]).max() < 1e-12
    F2 = oracle.force(a, L, m2, S, rho2)
    assert np.abs(F2 - F).max() < 1e-13


def test_translation_and_periodic_images(system):
    L, alpha, P, a, m, S, rho, F = system
    b = a.copy()
    b[:, :3] += np.float32(0.5)  # exact in fp32 on the 2^-12 grid
    Fb = oracle.force(b, L, m, S, oracle.rho(b, L, m))
    assert np.abs(Fb - F).max() < 1e-12
    c = a.copy()
    c[3, 0] += np.float32(L)
    c[7, 2] -= np.float32(2 * L)
    Fc = oracle.force(c, L, m, S, oracle.rho(c, L, m))
    assert np.abs(Fc - F).max() < 1e-12


def test_charge_scaling_and_permutation(system):
    L, alpha, P, a, m, S, rho, F = system
    b = a.copy()
    b[:, 3] *= np.float32(2.0)
    Fb = oracle.force(b, L, m, S, oracle.rho(b, L, m))
    assert np.abs(Fb - 4 * F).max() < 1e-12
    perm = np.random.default_rng(0).permutation(a.shape[0])
    Fp = oracle.force(a[perm], L, m, S, oracle.rho(a[perm], L, m))
    assert np.abs(Fp - F[perm]).max() < 1e-13


def test_selected_atoms_match_full(system):
    L, alpha, P, a, m, S, rho, F = system
    sel = np.array([49, 0, 17, 17, 3], dtype=np.int64)
    Fs, es = oracle.force(a, L, m, S, rho, sel=sel, with_energy=True)
    Ff, ef = oracle.force(a, L, m, S, rho, with_energy=True)
    assert np.array_equal(Fs, Ff[sel]) and np.array_equal(es, ef[sel])


# -------------------------------------------- deterministic limit: Eq. 2.11/2.8
def test_weighted_full_grid_is_exact_ewald():
    """With the k-set = every grid vector and w_l = exp(-k_l^2/4alpha) in place of Q/P,
    Eq. (2.12) IS Eq. (2.11) and the energy estimate IS the second term of Eq. (2.8)."""
    L, alpha, mmax = 6.0, 0.5, 7
    a = _atoms(12, L, 33)
    m = inputs.full_kgrid(mmax)
    k = _kvec(m, L)
    w = np.exp(-(k ** 2).sum(1) / (4 * alpha))
    rho = oracle.rho(a, L, m)
    F, e = oracle.force(a, L, m, 1.0, rho, w=w, with_energy=True)
    U = oracle.energy(L, m, 1.0, rho, w=w)
    Uref, _, Fl = oracle.ewald_full(a[:, :3].astype(np.float64), a[:, 3].astype(np.float64),
                                    L, alpha, nreal=0, mmax=mmax)
    assert np.abs(F - Fl).max() < 1e-13
    assert abs(U - Uref[1]) < 1e-13 * abs(Uref[1])
    assert abs(e.sum() - U) < 1e-13 * abs(U)


# ------------------------------------------------------ statistics
@pytest.fixture(scope="module")
def stat_system():
    L, alpha, mmax = 6.0, 0.5, 9
    a = _atoms(24, L, 77)
    r, q = a[:, :3].astype(np.float64), a[:, 3].astype(np.float64)
    Uref, _, Fl = oracle.ewald_full(r, q, L, alpha, nreal=0, mmax=mmax)
    return L, alpha, mmax, a, Uref[1], Fl


def _rbe_samples(a, L, alpha, P, T, seed):
    S = oracle.S(L, alpha)
    Fs = np.empty((T,) + (a.shape[0], 3))
    Us = np.empty(T)
    for t in range(T):
        m = inputs.sample_kset(L, alpha, P, seed, t)
        rho = oracle.rho(a, L, m)
        Fs[t] = oracle.force(a, L, m, S, rho)
        Us[t] = oracle.energy(L, m, S, rho)
    return Fs, Us


def test_unbiased_towards_exact_long_range_force(stat_system):
    """'the estimate (2.12) is unbiased': the mean over T seeds converges to Eq. (2.11)
    like 1/sqrt(T).  Catches any constant factor (S, 1/P, 4 pi, 1/V, 1/k^2) and the sign."""
    L, alpha, mmax, a, Uk, Fl = stat_system
    P, T = 20, 3000
    Fs, Us = _rbe_samples(a, L, alpha, P, T, 123)
    mean, sem = Fs.mean(0), Fs.std(0, ddof=1) / np.sqrt(T)
    z = (mean - Fl) / sem
    assert np.abs(z).max() < 5.0, np.abs(z).max()
    assert np.linalg.norm(mean - Fl) / np.linalg.norm(Fl) < 0.05
    # energy estimate: unbiased for the second term of Eq. (2.8)
    zu = (Us.mean() - Uk) / (Us.std(ddof=1) / np.sqrt(T))
    assert abs(zu) < 5.0, zu


def test_variance_closed_form_and_one_over_P(stat_system):
    """Var_total(P) = (1/P) [ S sum_k e^{-k^2/4alpha} |g(k)|^2 - |F_long|^2 ],
    g_i(k) = -(4 pi q_i k/(V k^2)) Im(e^{-ik.r_i} rho(k)): the 1/P law of P:133 with its constant."""
    L, alpha, mmax, a, Uk, Fl = stat_system
    S = oracle.S(L, alpha)
    m = inputs.full_kgrid(mmax)
    k = _kvec(m, L)
    k2 = (k ** 2).sum(1)
    r, q = a[:, :3].astype(np.float64), a[:, 3].astype(np.float64)
    ph = r @ k.T  # [N, K]
    rho = (q[:, None] * np.exp(1j * ph)).sum(0)
    im = np.imag(np.exp(-1j * ph) * rho[None, :])
    g = -(4 * np.pi / L ** 3) * q[:, None, None] * (k / k2[:, None])[None, :, :] * im[:, :, None]
    g2 = (g ** 2).sum((0, 2))
    base = S * (np.exp(-k2 / (4 * alpha)) * g2).sum() - (Fl ** 2).sum()
    ratios = []
    for P, T in [(10, 1500), (40, 1500), (160, 1000)]:
        Fs, _ = _rbe_samples(a, L, alpha, P, T, 1000 + P)
        var = Fs.var(0, ddof=1).sum()
        ratios.append(var / (base / P))
    assert all(abs(x - 1) < 0.12 for x in ratios), ratios
