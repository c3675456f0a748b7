"""Host-side checks of the seeded synthetic inputs (paper_2407_09315_b200/inputs.py):
BASELINE.json shapes/charges/geometry and the exact k-sampler (Algorithm 1 step 1)."""
import numpy as np
import pytest

from paper_2407_09315_b200 import inputs


@pytest.mark.parametrize("name", ["water_3k", "water_96k", "water_nacl_1m"])
def test_config_shapes_and_neutrality(name):
    cfg = inputs.CONFIGS[name]
    a = inputs.make_atoms(cfg)
    assert a.dtype == np.float32 and a.shape == (cfg.N, 4) and a.flags["C_CONTIGUOUS"]
    assert abs(cfg.N / cfg.L ** 3 - 0.1) < 5e-4  # 0.1 atoms / A^3 (BASELINE.json rounds L)
    assert abs(a[:, 3].astype(np.float64).sum()) < 1e-9  # exactly neutral in fp32
    assert np.array_equal(a, inputs.make_atoms(cfg))  # seeded, reproducible
    nw = cfg.n_water
    O, H1, H2 = (a[0:3 * nw:3, :3].astype(np.float64), a[1:3 * nw:3, :3].astype(np.float64),
                 a[2:3 * nw:3, :3].astype(np.float64))
    assert np.all(a[0:3 * nw:3, 3] == inputs.Q_O) and np.all(a[1:3 * nw:3, 3] == inputs.Q_H)
    d1, d2 = H1 - O, H2 - O
    assert np.abs(np.linalg.norm(d1, axis=1) - 1.0).max() < 1e-4  # |OH| = 1.0 A
    assert np.abs(np.linalg.norm(d2, axis=1) - 1.0).max() < 1e-4
    ang = np.degrees(np.arccos((d1 * d2).sum(1) / (np.linalg.norm(d1, axis=1) * np.linalg.norm(d2, axis=1))))
    assert np.abs(ang - 109.47).max() < 0.02
    assert O.min() >= 0 and O.max() < cfg.L
    # H atoms are deliberately not wrapped: some lie outside [0, L)
    H = np.concatenate([H1, H2])
    assert (H < 0).any() or (H >= cfg.L).any()


def test_nacl_reading_q13():
    """0.15 mol/L x V(L = 215.443 A) = 903 ion pairs; 332 731 waters + 1806 ions = 999 999."""
    cfg = inputs.CONFIGS["water_nacl_1m"]
    n_pairs = 0.15 * 6.02214076e23 * (cfg.L * 1e-9) ** 3  # L in dm = A * 1e-9
    assert round(n_pairs) == cfg.n_ion_pairs == 903
    assert 3 * cfg.n_water + 2 * cfg.n_ion_pairs == cfg.N == 999_999


def test_ion_sweep_boxes():
    for N, L in [(10 ** 4, 46.416), (10 ** 5, 100.0), (10 ** 6, 215.443), (10 ** 7, 464.159), (10 ** 8, 1000.0)]:
        assert abs(inputs.ion_box(N) - L) < 1e-3
    cfg = inputs.ions_config(10 ** 4)
    a = inputs.make_atoms(cfg)
    assert a.shape == (10 ** 4, 4) and a[:, 3].sum() == 0 and set(np.unique(a[:, 3])) == {-1.0, 1.0}


def test_sampler_distribution():
    """chi^2 of the m_d histogram against the 1-D pmf conditional on m != 0; no zero vector;
    second moment E[m_d^2] ~ alpha L^2 / (2 pi^2)."""
    L, alpha, P = 31.04, 0.09, 200_000
    m = inputs.sample_kset(L, alpha, P, seed=7, step=3)
    assert m.dtype == np.int32 and m.shape == (P, 3)
    assert np.all(np.any(m != 0, axis=1))
    ms, p = inputs.pmf_1d(L, alpha)
    p0 = p[ms == 0][0]
    # marginal of one component given the triple is not (0,0,0)
    marg = p.copy()
    marg[ms == 0] = p0 * (1 - p0 * p0)
    marg[ms != 0] = p[ms != 0]
    marg /= (1 - p0 ** 3)
    assert abs(marg.sum() - 1) < 1e-12
    for d in range(3):
        big = marg * P >= 20
        obs = np.array([(m[:, d] == v).sum() for v in ms[big]])
        chi2 = ((obs - marg[big] * P) ** 2 / (marg[big] * P)).sum()
        dof = big.sum() - 1
        assert chi2 < dof + 6 * np.sqrt(2 * dof), (d, chi2, dof)
    sigma2 = alpha * L * L / (2 * np.pi ** 2)
    emp = (m.astype(np.float64) ** 2).mean()
    assert abs(emp / (sigma2 / (1 - p0 ** 3)) - 1) < 0.02


def test_sampler_seeding():
    a = inputs.sample_kset(98.65, 0.09, 100, 2, 0)
    assert np.array_equal(a, inputs.sample_kset(98.65, 0.09, 100, 2, 0))
    assert not np.array_equal(a, inputs.sample_kset(98.65, 0.09, 100, 2, 1))
    assert np.abs(a).max() < 2 ** 15


def test_full_kgrid_and_shards():
    g = inputs.full_kgrid(2)
    assert g.shape == (124, 3) and np.all(np.any(g != 0, axis=1))
    N = 999_999
    for ws in (1, 2, 3, 8):
        edges = [inputs.shard_bounds(N, ws, r, align=32) for r in range(ws)]
        assert edges[0][0] == 0 and edges[-1][1] == N
        for (a0, a1), (b0, b1) in zip(edges[:-1], edges[1:]):
            assert a1 == b0 and a1 % 32 == 0
        sizes = [hi - lo for lo, hi in edges]
        assert max(sizes) - min(sizes) <= 64
