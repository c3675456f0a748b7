"""Fused multi-GPU exchange of the structure factors (rbe_set_exchange), exercised on ONE device.

Several contexts play the ranks; their exchange buffers live on the same GPU, which is exactly
what a rank sees of its peers' buffers over NVLink (plain global addresses).  The launches are
ordered so that every push has completed before any consumer runs (all structure-factor launches
first, then the force launches, on one stream): no kernel ever waits for a kernel that has not
been launched, as the profiling guide requires on a single GPU."""
import numpy as np
import pytest
import torch

import oracle
from paper_2407_09315_b200 import inputs, rbe

pytestmark = pytest.mark.gpu


def _ranks(cfg, atoms, world):
    ctxs, xs, bufs = [], [], []
    for r in range(world):
        lo, hi = inputs.shard_bounds(cfg.N, world, r, align=32)
        xs.append(torch.from_numpy(atoms[lo:hi].copy()).cuda())
        ctxs.append(rbe.Rbe(hi - lo, cfg.L, cfg.alpha, cfg.P))
    nbytes = ctxs[0].rbe_exchange_bytes(world)
    assert nbytes >= 2 * world * cfg.P * 16 + 2 * world * 4
    bufs = [torch.zeros(nbytes, dtype=torch.uint8, device="cuda") for _ in range(world)]
    for r, c in enumerate(ctxs):
        c.rbe_set_exchange(r, world, [b.data_ptr() for b in bufs], nbytes, keep_alive=bufs)
    return ctxs, xs, bufs


@pytest.mark.parametrize("world", [2, 3])
def test_fused_exchange_matches_oracle_and_injected_sum(world):
    cfg = inputs.CONFIGS["water_96k"]
    atoms = inputs.make_atoms(cfg)
    ctxs, xs, bufs = _ranks(cfg, atoms, world)
    S = oracle.S(cfg.L, cfg.alpha)
    for step in range(3):                      # both parities of the slots, and their reuse
        m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, step)
        parts = [torch.empty((cfg.P, 2), dtype=torch.float64, device="cuda") for _ in range(world)]
        for c, x, part in zip(ctxs, xs, parts):
            c.rbe_set_kvectors(m)
            c.rbe_structure_factor(x, part)     # pushes the partial into every rank's buffer
        Fs, Us = [], []
        for c, x in zip(ctxs, xs):
            F = torch.empty((x.shape[0], 4), dtype=torch.float32, device="cuda")
            c.rbe_forces(x, F, True)
            Fs.append(F)
            Us.append(c.rbe_kspace_energy())
            c.rbe_exchange_check()
        # reference data path: rank-ordered sum injected with rbe_set_rho into exchange-free contexts
        total = torch.zeros_like(parts[0])
        for part in parts:
            total = total + part
        for r, x in enumerate(xs):
            ref = rbe.Rbe(x.shape[0], cfg.L, cfg.alpha, cfg.P)
            ref.rbe_set_kvectors(m)
            ref.rbe_set_rho(total)
            Fr = torch.empty_like(Fs[r])
            ref.rbe_forces(x, Fr, True)
            assert torch.equal(Fs[r], Fr)                       # bitwise: same rho, same kernel
            assert ref.rbe_kspace_energy() == Us[r]
        assert len(set(Us)) == 1                                # every rank sees the same global rho
        rho_o = oracle.rho(atoms, cfg.L, m)
        F_o = oracle.force(atoms, cfg.L, m, S, rho_o)
        F_g = torch.cat(Fs).cpu().numpy()[:, :3].astype(np.float64)
        assert np.abs(total.cpu().numpy() - rho_o).max() <= 1e-6 * np.abs(atoms[:, 3]).sum()
        assert np.linalg.norm(F_g - F_o) / np.linalg.norm(F_o) <= 2e-5
        assert abs(Us[0] - oracle.energy(cfg.L, m, S, rho_o)) <= 1e-5 * abs(Us[0])


def test_exchange_argument_checks_and_exclusions():
    cfg = inputs.CONFIGS["water_3k"]
    ctx = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
    n = ctx.rbe_exchange_bytes(2)
    buf = torch.zeros(n, dtype=torch.uint8, device="cuda")
    assert ctx.rbe_exchange_bytes(0) == 0 and ctx.rbe_exchange_bytes(17) == 0
    with pytest.raises(rbe.RbeError):
        ctx.rbe_set_exchange(2, 2, [buf.data_ptr(), buf.data_ptr()], n)      # rank out of range
    with pytest.raises(rbe.RbeError):
        ctx.rbe_set_exchange(0, 2, [buf.data_ptr(), buf.data_ptr()], n - 1)  # too small
    with pytest.raises(rbe.RbeError):
        ctx.rbe_set_exchange(0, 2, [buf.data_ptr(), buf.data_ptr() + 8], n)  # misaligned
    ctx.rbe_set_exchange(0, 1, [buf.data_ptr()], n, keep_alive=buf)          # a world of one: push to self
    x = torch.from_numpy(inputs.make_atoms(cfg)).cuda()
    F = torch.empty((cfg.N, 4), dtype=torch.float32, device="cuda")
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    ctx.rbe_set_kvectors(m)
    rho = torch.empty((cfg.P, 2), dtype=torch.float64, device="cuda")
    ctx.rbe_structure_factor(x, rho)
    with pytest.raises(rbe.RbeError):
        ctx.rbe_set_rho(rho)
    with pytest.raises(rbe.RbeError):
        ctx.rbe_graph_capture(x, F, False, 1, 0)
    ctx.rbe_forces(x, F)
    ctx.rbe_exchange_check()
    ctx.rbe_set_exchange(0, 0, None, 0)                                       # off again
    ref = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
    ref.rbe_set_kvectors(m)
    ref.rbe_structure_factor(x)
    Fr = torch.empty_like(F)
    ref.rbe_forces(x, Fr)
    assert torch.equal(F, Fr)


def test_symmetric_memory_plumbing_world_of_one():
    """paper_2407_09315_b200.exchange.setup_fused_exchange on a one-rank NCCL group: the buffer is a
    real torch symmetric-memory allocation and the kernels push to / pull from it."""
    import os
    import torch.distributed as dist
    from paper_2407_09315_b200 import exchange
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        os.environ["MASTER_PORT"] = str(sk.getsockname()[1])
    created = not dist.is_initialized()
    if created:
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        cfg = inputs.CONFIGS["water_3k"]
        atoms = inputs.make_atoms(cfg)
        x = torch.from_numpy(atoms).cuda()
        ctx = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
        exchange.setup_fused_exchange(ctx)
        ref = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
        for step in range(3):
            m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, step)
            F, Fr = (torch.empty((cfg.N, 4), dtype=torch.float32, device="cuda") for _ in range(2))
            for c, out in ((ctx, F), (ref, Fr)):
                c.rbe_set_kvectors(m)
                c.rbe_structure_factor(x)
                c.rbe_forces(x, out, True)
            ctx.rbe_exchange_check()
            assert torch.equal(F, Fr) and ctx.rbe_kspace_energy() == ref.rbe_kspace_energy()
    finally:
        if created:
            dist.destroy_process_group()
