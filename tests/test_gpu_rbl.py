"""Parity of the random batch list on the GPU (rbe_rbl_forces) against oracle/rbl.py: the batch is decided
by integer keys (a salted hash, reading Q20), so both sides pick the same neighbours and the forces agree to the fp32 pair
arithmetic (2e-5 relative L2, the bar of the deterministic short-range force)."""
import numpy as np
import pytest
import torch

import oracle
from oracle import rbl as orbl
from paper_2407_09315_b200 import inputs, rbe

pytestmark = pytest.mark.gpu


def gpu_rbl(atoms, L, alpha, rc, rs, p, seed, step, base=None):
    N = atoms.shape[0]
    ctx = rbe.Rbe(N, L, alpha, 4, allocate=False)
    x = torch.from_numpy(atoms).cuda()
    F = torch.full((N, 4), float("nan"), dtype=torch.float32, device="cuda") if base is None else base.clone()
    ctx.rbe_rbl_forces(x, rc, rs, p, seed, step, F, accumulate=base is not None)
    torch.cuda.synchronize()
    return ctx, x, F


@pytest.mark.parametrize("name,rc,rs,p", [("water_3k", 5.0, 10.0, 30), ("water_3k", 4.0, 8.0, 8), ("ions_4000", 6.0, 11.0, 32)])
def test_rbl_matches_oracle(name, rc, rs, p):
    cfg = inputs.CONFIGS[name] if name in inputs.CONFIGS else inputs.ions_config(4000)
    atoms = inputs.make_atoms(cfg)
    for step in (0, (1 << 33) + 5):
        _, _, F = gpu_rbl(atoms, cfg.L, cfg.alpha, rc, rs, p, seed=(1 << 40) + 11, step=step)
        Fg = F.cpu().numpy().astype(np.float64)
        F_o, Ns, Fc = orbl.rbl_forces(atoms, cfg.L, cfg.alpha, rc, rs, p, (1 << 40) + 11, step)
        assert Ns.min() > p                                                   # the random branch everywhere
        assert np.isfinite(Fg).all() and np.all(Fg[:, 3] == 0)
        assert np.linalg.norm(Fg[:, :3] - F_o) / np.linalg.norm(F_o) <= 2e-5
        assert np.abs(Fg[:, :3].sum(0)).max() <= 1e-5 * np.abs(Fg[:, :3]).sum()   # Eq. 2.16: momentum conserved


def test_rbl_with_the_whole_shell_equals_the_deterministic_kernel():
    cfg = inputs.CONFIGS["water_3k"]
    atoms = inputs.make_atoms(cfg)
    rc, rs = 2.5, 6.0                                   # N_s ~ 88 > 32, so shrink the shell instead: r_c close to r_s
    rc = 5.8
    _, _, F = gpu_rbl(atoms, cfg.L, cfg.alpha, rc, rs, 32, 1, 0)
    F_o, Ns, _ = orbl.rbl_forces(atoms, cfg.L, cfg.alpha, rc, rs, 32, 1, 0)
    assert Ns.max() <= 32                                # every shell fits the batch: nothing random is left
    Fd, _ = oracle.short_range(atoms, cfg.L, cfg.alpha, rs)
    Fg = F.cpu().numpy()[:, :3].astype(np.float64)
    assert np.linalg.norm(Fg - Fd) / np.linalg.norm(Fd) <= 2e-5
    assert np.linalg.norm(Fg - F_o) / np.linalg.norm(F_o) <= 2e-5


def test_rbl_reproducible_accumulate_and_argument_checks():
    cfg = inputs.CONFIGS["water_3k"]
    atoms = inputs.make_atoms(cfg)
    ctx, x, F1 = gpu_rbl(atoms, cfg.L, cfg.alpha, 5.0, 10.0, 30, 3, 9)
    _, _, F2 = gpu_rbl(atoms, cfg.L, cfg.alpha, 5.0, 10.0, 30, 3, 9)
    assert torch.equal(F1, F2)
    _, _, F3 = gpu_rbl(atoms, cfg.L, cfg.alpha, 5.0, 10.0, 30, 3, 10)
    assert not torch.equal(F1, F3)
    base = torch.ones((cfg.N, 4), dtype=torch.float32, device="cuda")
    _, _, F4 = gpu_rbl(atoms, cfg.L, cfg.alpha, 5.0, 10.0, 30, 3, 9, base=base)
    assert torch.allclose(F4[:, :3], F1[:, :3] + 1.0, rtol=0, atol=1e-6) and torch.all(F4[:, 3] == 1.0)
    for bad in [(0.0, 10.0, 30), (10.0, 10.0, 30), (5.0, 10.0, 0), (5.0, 10.0, 33), (5.0, cfg.L / 2.9, 30)]:
        with pytest.raises(rbe.RbeError):
            ctx.rbe_rbl_forces(x, bad[0], bad[1], bad[2], 1, 1, F1)


@pytest.mark.parametrize("kind", ["blob", "dense"])
def test_rbl_list_free_path_for_crowded_atoms_and_cells(kind):
    """The fast path keeps an atom's hits in fixed-size per-lane columns and a cell's candidates in a fixed-size
    tile; anything that does not fit takes the list-free path (bisection on the key threshold).  'blob': 1200 atoms
    inside a 9 A ball (hundreds of shell members per lane column); 'dense': 0.2 atoms/A^3 everywhere (the 125-cell
    candidate set exceeds the tile).  Same oracle, same bar."""
    rng = np.random.default_rng(17)
    L, alpha = 31.0, 0.09
    if kind == "blob":
        n_bg, n_blob = 1500, 1200
        pos = rng.random((n_bg, 3)) * L
        v = rng.standard_normal((n_blob, 3))
        v *= (4.5 * rng.random((n_blob, 1)) ** (1 / 3)) / np.linalg.norm(v, axis=1, keepdims=True)
        pos = np.concatenate([pos, v + L / 2])
    else:
        pos = rng.random((6000, 3)) * L
    atoms = np.empty((pos.shape[0], 4), dtype=np.float32)
    atoms[:, :3] = pos
    atoms[:, 3] = np.where(np.arange(pos.shape[0]) % 2 == 0, 1.0, -1.0)
    rc, rs, p = 4.0, 8.0, 16
    _, _, F = gpu_rbl(atoms, L, alpha, rc, rs, p, seed=5, step=2)
    _, _, F2 = gpu_rbl(atoms, L, alpha, rc, rs, p, seed=5, step=2)
    assert torch.equal(F, F2)
    Fg = F.cpu().numpy().astype(np.float64)
    F_o, Ns, _ = orbl.rbl_forces(atoms, L, alpha, rc, rs, p, 5, 2)
    assert Ns.max() > (400 if kind == "blob" else 300)
    assert np.isfinite(Fg).all()
    assert np.linalg.norm(Fg[:, :3] - F_o) / np.linalg.norm(F_o) <= 2e-5
