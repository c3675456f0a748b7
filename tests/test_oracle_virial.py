"""Pin of oracle/virial.py (reading Q19): the k-space virial is minus the strain derivative
of the second term of Eq. (2.8) P:112.  The energy of an orthorhombic (and, for the off-diagonal
components, sheared) periodic cell is written out here from its definition and differentiated by
central differences; the oracle's closed form must agree component by component."""
import itertools

import numpy as np

import oracle
from oracle import virial
from paper_2407_09315_b200 import inputs


def _uk_general(r, q, H, alpha, mmax):
    """U_k = (2 pi / V) sum_{m != 0} |rho(k)|^2 exp(-k^2/4alpha) / k^2,  k = 2 pi H^{-T} m, for a cell matrix H."""
    V = abs(np.linalg.det(H))
    G = 2.0 * np.pi * np.linalg.inv(H).T            # columns of H are the cell vectors
    U = 0.0
    for mm in itertools.product(range(-mmax, mmax + 1), repeat=3):
        if mm == (0, 0, 0):
            continue
        k = G @ np.array(mm, dtype=np.float64)
        k2 = k @ k
        ph = r @ k
        re, im = (q * np.cos(ph)).sum(), (q * np.sin(ph)).sum()
        U += 2.0 * np.pi / V * (re * re + im * im) * np.exp(-k2 / (4.0 * alpha)) / k2
    return U


def test_virial_is_minus_the_strain_derivative_of_the_kspace_energy():
    L, alpha, mmax, n = 9.0, 0.5, 6, 10
    rng = np.random.default_rng(5)
    r = rng.random((n, 3)) * L
    q = np.where(np.arange(n) % 2 == 0, 1.0, -1.0) * (0.5 + rng.random(n))
    m = inputs.full_kgrid(mmax)
    k2 = (2 * np.pi / L) ** 2 * (m.astype(np.float64) ** 2).sum(1)
    w = np.exp(-k2 / (4 * alpha))
    xyzq = np.concatenate([r, q[:, None]], axis=1).astype(np.float32)
    r, q = xyzq[:, :3].astype(np.float64), xyzq[:, 3].astype(np.float64)     # what the oracle sees
    rho = oracle.rho(xyzq, L, m)
    W = virial.kspace_virial(L, alpha, m, 0.0, rho, w=w)
    # energy consistency: the closed form and the written-out sum describe the same U
    assert abs(oracle.energy(L, m, 0.0, rho, w=w) - _uk_general(r, q, np.eye(3) * L, alpha, mmax)) < 1e-12
    h = 1e-5
    for idx, (a, b) in enumerate(((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2))):
        def U(e):
            eps = np.zeros((3, 3))
            eps[a, b] += e / 2
            eps[b, a] += e / 2                        # symmetric strain; for a == b this is eps_aa = e
            D = np.eye(3) + eps
            return _uk_general(r @ D.T, q, D @ (np.eye(3) * L), alpha, mmax)
        dU = (U(h) - U(-h)) / (2 * h)
        assert abs(-dU - W[idx]) <= 1e-7 * np.abs(W).max(), (a, b, -dU, W[idx])
    # trace identity: tr W = U_k - (1 / 2 alpha) (2 pi / V) sum_k g |rho|^2
    Uk = oracle.energy(L, m, 0.0, rho, w=w)
    extra = (2 * np.pi / L ** 3 * w * (rho ** 2).sum(1)).sum() / (2 * alpha)
    assert abs(W[:3].sum() - (Uk - extra)) <= 1e-12 * abs(Uk)


def test_rbe_weights_and_symmetries():
    cfg = inputs.CONFIGS["water_3k"]
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    S = oracle.S(cfg.L, cfg.alpha)
    rho = oracle.rho(atoms, cfg.L, m)
    W = virial.kspace_virial(cfg.L, cfg.alpha, m, S, rho)
    Wm = virial.kspace_virial(cfg.L, cfg.alpha, -m, S, rho * [1, -1])        # k -> -k: rho -> conj(rho)
    assert np.allclose(W, Wm, rtol=1e-14, atol=0)
    perm = [1, 2, 0]                                                           # relabel the axes
    Wp = virial.kspace_virial(cfg.L, cfg.alpha, m[:, perm], S, rho)
    assert np.allclose(Wp[:3], W[[1, 2, 0]], rtol=1e-14) and np.allclose(Wp[3:], W[[5, 3, 4]], rtol=1e-13)
    assert np.allclose(virial.kspace_virial(cfg.L, cfg.alpha, m, S, rho, w=np.full(cfg.P, S / cfg.P)), W, rtol=1e-15)
