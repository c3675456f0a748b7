"""Device sampler (Algorithm 1 step 1 on the GPU, bit-exact against oracle/sampler.py) and the
graph-captured whole step (sampler + structure factor + force in one launch)."""
import numpy as np
import pytest
import torch

import oracle
from oracle import sampler as osampler
from paper_2407_09315_b200 import inputs, rbe

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("L,alpha,P,seed,step", [
    (31.04, 0.09, 100, 1, 0),
    (215.443, 0.09, 200, 3, 17),
    (6.0, 0.3, 200, 7, 3),                     # zero triples are frequent: the rejection rule matters
    (1000.0, 0.09, 1600, 5, (1 << 40) + 3),    # widest table of the sweep; high word of the step
    (98.65, 0.09, 5000, (1 << 35) + 9, 2),     # several 1024-candidate rounds; high word of the seed
    (4.0, 0.05, 1, 2, 2),                      # M = 1: the smallest table; P = 1
])
def test_device_sampler_is_bit_exact(L, alpha, P, seed, step):
    ctx = rbe.Rbe(64, L, alpha, P)
    ctx.rbe_sample_kvectors(seed, step)
    got = ctx.rbe_get_kvectors()
    want = osampler.sample_kset(L, alpha, P, seed, step)
    assert got.dtype == np.int32 and np.array_equal(got, want)
    assert np.all(np.any(got != 0, axis=1))


def test_sampled_step_matches_oracle_and_host_fed_path():
    cfg = inputs.CONFIGS["water_96k"]
    atoms = inputs.make_atoms(cfg)
    x = torch.from_numpy(atoms).cuda()
    F1 = torch.empty((cfg.N, 4), dtype=torch.float32, device="cuda")
    F2 = torch.empty_like(F1)
    ctx = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
    ctx.rbe_sample_kvectors(42, 5)
    ctx.rbe_structure_factor(x)
    ctx.rbe_forces(x, F1, True)
    U1 = ctx.rbe_kspace_energy()
    m = osampler.sample_kset(cfg.L, cfg.alpha, cfg.P, 42, 5)
    ctx.rbe_set_kvectors(m)                       # the same batch handed over from the host
    ctx.rbe_structure_factor(x)
    ctx.rbe_forces(x, F2, True)
    assert torch.equal(F1, F2) and ctx.rbe_kspace_energy() == U1
    S = oracle.S(cfg.L, cfg.alpha)
    rho_o = oracle.rho(atoms, cfg.L, m)
    F_o = oracle.force(atoms, cfg.L, m, S, rho_o)
    assert np.linalg.norm(F1.cpu().numpy()[:, :3] - F_o) / np.linalg.norm(F_o) <= 2e-5
    assert abs(U1 - oracle.energy(cfg.L, m, S, rho_o)) <= 1e-5 * abs(U1)


@pytest.mark.parametrize("name", ["water_3k", "water_96k"])
def test_graph_replay_advances_the_step_and_matches_separate_launches(name):
    cfg = inputs.CONFIGS[name]
    atoms = inputs.make_atoms(cfg)
    x = torch.from_numpy(atoms).cuda()
    Fg = torch.full((cfg.N, 4), float("nan"), dtype=torch.float32, device="cuda")
    Fs = torch.empty_like(Fg)
    ctx = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
    ref = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
    with pytest.raises(rbe.RbeError):
        ctx.rbe_graph_launch()
    ctx.rbe_graph_capture(x, Fg, True, seed=9, first_step=5)
    S = oracle.S(cfg.L, cfg.alpha)
    for step in (5, 6, 7):
        ctx.rbe_graph_launch()
        torch.cuda.synchronize()
        m = ctx.rbe_get_kvectors()
        assert np.array_equal(m, osampler.sample_kset(cfg.L, cfg.alpha, cfg.P, 9, step))
        ref.rbe_sample_kvectors(9, step)
        ref.rbe_step(None, x, Fs, with_energy=True)            # the same kernels outside the graph: bitwise equal
        assert torch.equal(Fg, Fs)
        assert ctx.rbe_kspace_energy() == ref.rbe_kspace_energy()
        ref.rbe_structure_factor(x)                            # the two-launch form: another fixed order of the rows and
        ref.rbe_forces(x, Fs, True)                            # fp64 instead of fp32 atan2 in the per-k records
        assert torch.allclose(Fg, Fs, rtol=0, atol=2e-5 * float(Fs[:, :3].abs().max()))
        rho_o = oracle.rho(atoms, cfg.L, m)
        F_o = oracle.force(atoms, cfg.L, m, S, rho_o)
        assert np.linalg.norm(Fg.cpu().numpy()[:, :3] - F_o) / np.linalg.norm(F_o) <= 2e-5
    # positions may change between replays (the graph is bound to the buffer, not its contents)
    x.add_(0.25)
    ctx.rbe_graph_launch()
    ref.rbe_sample_kvectors(9, 8)
    ref.rbe_step(None, x, Fs, with_energy=True)
    assert torch.equal(Fg, Fs)


def test_mean_of_graph_replays_converges_to_the_deterministic_ewald_force():
    """End to end on the device (sampler + structure factor + force, one graph launch per step): the RBE
    force is an unbiased estimator of Eq. (2.11), so the mean over T replays approaches the
    full k-space force of oracle.ewald_full like 1/sqrt(T); the residual after T and 4T steps must
    shrink by about 2, and be consistent with the closed-form variance (~ 1/P)."""
    L, alpha, P = 20.0, 0.25, 50
    cfg = inputs.ions_config(400)
    atoms = inputs.make_atoms(cfg)
    atoms[:, :3] *= np.float32(L / cfg.L)
    x = torch.from_numpy(atoms).cuda()
    F = torch.empty((400, 4), dtype=torch.float32, device="cuda")
    ctx = rbe.Rbe(400, L, alpha, P)
    ctx.rbe_graph_capture(x, F, False, seed=77, first_step=0)
    _, _, F_long = oracle.ewald_full(atoms[:, :3].astype(np.float64), atoms[:, 3].astype(np.float64), L, alpha, nreal=0, mmax=14)
    acc = torch.zeros((400, 3), dtype=torch.float64, device="cuda")
    sq = torch.zeros((), dtype=torch.float64, device="cuda")
    res = {}
    for t in range(1, 1601):
        ctx.rbe_graph_launch()
        f = F[:, :3].double()
        acc += f
        sq += (f * f).sum()
        if t in (400, 1600):
            res[t] = np.linalg.norm((acc / t).cpu().numpy() - F_long)
    nrm = np.linalg.norm(F_long)
    # variance of one step's estimate (summed over components), measured, predicts the residual of the mean
    var1 = float(sq.item()) / 1600 - float(((acc / 1600) ** 2).sum().item())
    # (the per-step error is heavy-tailed -- rare small-|k| samples carry large weights -- so the typical
    # residual sits below its rms expectation; a bias would show as a floor that does not shrink)
    for t in (400, 1600):
        expect = np.sqrt(var1 / t)
        assert 0.4 * expect <= res[t] <= 1.5 * expect, (t, res[t], expect)
    assert 1.4 <= res[400] / res[1600] <= 2.8, res
    assert res[1600] <= 0.2 * nrm
