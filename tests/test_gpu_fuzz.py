"""Randomised parity sweep (fixed seed): sizes, boxes, splitting parameters, charge patterns, pairing
modes and cutoffs drawn at random; the device sampler must reproduce the oracle's batch bit for bit, and
rho, forces, energy, short-range forces and RBL forces must meet the usual bars.  Where a force vanishes
by cancellation (N = 1, zero charges) or falls below the fixed-point resolution of the short-range
accumulators, the error is measured against the natural scale of its terms instead of its own norm.
(A longer run of the same sweep caught the absolutely-but-not-relatively accurate erfc of the first
short-range kernel.)"""
import numpy as np
import pytest
import torch

import oracle
from oracle import rbl as orbl
from oracle import sampler as osampler
from paper_2407_09315_b200 import rbe

pytestmark = pytest.mark.gpu


def _case(rng):
    N = int(rng.choice([rng.integers(1, 200), rng.integers(200, 3000), rng.integers(3000, 40000)]))
    P = int(rng.choice([rng.integers(1, 40), rng.integers(40, 400), rng.integers(400, 2600)]))
    L, alpha = float(rng.uniform(8, 300)), float(rng.uniform(0.03, 0.6))
    atoms = np.empty((N, 4), dtype=np.float32)
    atoms[:, :3] = (rng.random((N, 3)) * L * rng.choice([1.0, 1.0, 7.0]) - rng.choice([0.0, 3.0 * L])).astype(np.float32)
    kind = int(rng.integers(0, 4))
    if kind == 0:
        atoms[:, 3] = np.where(np.arange(N) % 2 == 0, 1.0, -1.0)
    elif kind == 1:
        atoms[:, 3] = rng.choice(np.array([-0.8476, 0.4238, 0.4238], dtype=np.float32), N)
    elif kind == 2:
        atoms[:, 3] = (rng.random(N) * 2 - 1).astype(np.float32)
    else:
        atoms[:, 3] = rng.choice(np.array([0.0, 1.0, -1.0, 2.0, -0.5], dtype=np.float32), N)
    return N, P, L, alpha, atoms


def test_randomised_parity_sweep():
    rng = np.random.default_rng(2024)
    for it in range(60):
        N, P, L, alpha, atoms = _case(rng)
        seed, step = int(rng.integers(0, 2 ** 40)), int(rng.integers(0, 2 ** 40))
        tag = dict(it=it, N=N, P=P, L=L, alpha=alpha, seed=seed, step=step)
        ctx = rbe.Rbe(N, L, alpha, P)
        ctx.rbe_set_pairing(int(rng.choice([0, 1, 3])))
        x = torch.from_numpy(atoms).cuda()
        F = torch.full((N, 4), float("nan"), dtype=torch.float32, device="cuda")
        rho = torch.empty((P, 2), dtype=torch.float64, device="cuda")
        ctx.rbe_sample_kvectors(seed, step)
        m = ctx.rbe_get_kvectors()
        assert np.array_equal(m, osampler.sample_kset(L, alpha, P, seed, step)), tag
        ctx.rbe_structure_factor(x, rho)
        ctx.rbe_forces(x, F, bool(rng.integers(0, 2)))
        U = ctx.rbe_kspace_energy()
        S = oracle.S(L, alpha)
        rho_o = oracle.rho(atoms, L, m)
        q = atoms[:, 3].astype(np.float64)
        assert np.abs(rho.cpu().numpy() - rho_o).max() <= 1e-6 * max(np.abs(q).sum(), 1e-300), tag
        F_o = oracle.force(atoms, L, m, S, rho_o)
        Fg = F.cpu().numpy().astype(np.float64)
        assert np.isfinite(Fg).all(), tag
        k2 = (2 * np.pi / L) ** 2 * (m.astype(np.float64) ** 2).sum(1)
        term = 4 * np.pi * S / (L ** 3 * P) / np.sqrt(k2) * np.hypot(rho_o[:, 0], rho_o[:, 1])     # |c_l| |rho_l|
        scale = np.linalg.norm(q) * term.sum()
        assert np.linalg.norm(Fg[:, :3] - F_o) <= 2e-5 * np.linalg.norm(F_o) + 1e-7 * scale, tag
        U_o = oracle.energy(L, m, S, rho_o)
        assert abs(U - U_o) <= 1e-5 * abs(U_o) + 1e-300, tag
        if N <= 4000:
            rs = float(rng.uniform(0.15, 0.33) * L)
            Fs = torch.full((N, 4), float("nan"), dtype=torch.float32, device="cuda")
            ctx.rbe_short_range(x, rs, Fs, with_energy=True)
            Fs_o, _ = oracle.short_range(atoms, L, alpha, rs)
            Fsg = Fs.cpu().numpy().astype(np.float64)
            floor = 1e-11 * np.sqrt(N) * max(np.abs(q).max(), 1e-300)       # fixed-point resolution of the accumulators
            assert np.isfinite(Fsg).all(), tag
            assert np.linalg.norm(Fsg[:, :3] - Fs_o) <= 2e-5 * np.linalg.norm(Fs_o) + floor, (tag, rs)
            for kind, table in ((0, True), (1, False), (1, True)):          # the other force kernel / the tabulated pair term
                ctx.rbe_set_pair_kernel(kind)
                ctx.rbe_set_pair_table(table)
                Fv = torch.full((N, 4), float("nan"), dtype=torch.float32, device="cuda")
                ctx.rbe_short_range(x, rs, Fv, with_energy=True)
                Fvg = Fv.cpu().numpy().astype(np.float64)
                assert np.isfinite(Fvg).all(), (tag, kind, table)
                assert np.linalg.norm(Fvg[:, :3] - Fs_o) <= 2e-5 * np.linalg.norm(Fs_o) + floor, (tag, rs, kind, table)
            ctx.rbe_set_pair_kernel(0)
            ctx.rbe_set_pair_table(False)
            if 2 <= N <= 1200:
                p, rc = int(rng.integers(1, 33)), float(rng.uniform(0.3, 0.8) * rs)
                Fr = torch.full((N, 4), float("nan"), dtype=torch.float32, device="cuda")
                ctx.rbe_rbl_forces(x, rc, rs, p, seed, step, Fr)
                Fr_o, _, _ = orbl.rbl_forces(atoms, L, alpha, rc, rs, p, seed, step)
                Frg = Fr.cpu().numpy().astype(np.float64)
                assert np.linalg.norm(Frg[:, :3] - Fr_o) <= 2e-5 * np.linalg.norm(Fr_o) + 40 * floor, (tag, rc, rs, p)
