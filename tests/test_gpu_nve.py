"""The NVE velocity-Verlet loop on the GPU (rbe_nve_kick, rbe_md_capture) against
oracle/nve.py over 100 steps of a perturbed rock-salt crystal (216 ions).

Tolerance (paper silent; derived).  Both sides keep x, v in fp64 and evaluate the forces on fp32-rounded
positions; the GPU forces carry ~1e-6 relative error (fp32 pair arithmetic), i.e. ~3e-7 e^2/A^2 per ion and
step.  A velocity error of dt/2m * dF ~ 3e-9 A/tau per step random-walks to ~3e-8 over 100 steps and the
positions to ~1e-6 A; the crystal is a saddle point of the pure Coulomb energy (nothing but the short horizon
keeps unlike charges apart), which amplifies differences by ~e^3 over these 20 tau.
Bars: 1e-4 A on positions, 2e-5 A/tau on velocities (0.3 % of the thermal velocity), 2e-6 relative on energy."""
import numpy as np
import pytest
import torch

import oracle
from oracle import nve as onve
from oracle import sampler as osampler
from paper_2407_09315_b200 import inputs, rbe

pytestmark = pytest.mark.gpu

DT, NSTEPS = 0.2, 100


def _system():
    x, v, q, mass, L = inputs.rocksalt(3, seed=11, jitter=0.05, v_rms=0.04)
    rs = L / 3.0
    alpha = (3.4 / rs) ** 2
    return x, v, q, mass, L, alpha, rs


def _gpu_state(x, v, q, mass):
    pos = torch.from_numpy(x.copy()).cuda()
    vel = torch.from_numpy(v.copy()).cuda()
    inv_m = torch.from_numpy(1.0 / mass).cuda()
    xyzq = torch.from_numpy(np.concatenate([x.astype(np.float32), q[:, None]], axis=1)).cuda().contiguous()
    force = torch.zeros((x.shape[0], 4), dtype=torch.float32, device="cuda")
    return pos, vel, inv_m, xyzq, force


def _energy(ctx, vel, inv_m, force, q, alpha):
    ke, uw = ctx.rbe_nve_energies(vel, inv_m, force)
    return ke + uw - np.sqrt(alpha / np.pi) * float((q.astype(np.float64) ** 2).sum())


def test_deterministic_ewald_trajectory_matches_the_oracle():
    x, v, q, mass, L, alpha, rs = _system()
    mmax = int(np.ceil(np.sqrt(18.4 * 4 * alpha) * L / (2 * np.pi)))
    m = inputs.full_kgrid(mmax)
    w = np.exp(-(2 * np.pi / L) ** 2 * (m.astype(np.float64) ** 2).sum(1) / (4 * alpha))
    xs, vs, Es = onve.run(x, v, q, mass, L, alpha, rs, DT, NSTEPS, m, w)

    ctx = rbe.Rbe(x.shape[0], L, alpha, m.shape[0])
    pos, vel, inv_m, xyzq, force = _gpu_state(x, v, q, mass)
    ctx.rbe_set_kvectors(m, w)

    def forces():
        ctx.rbe_step(None, xyzq, force, with_energy=True)
        ctx.rbe_short_range(xyzq, rs, force, accumulate=True, with_energy=True)

    # (a) explicit calls: kick + drift, forces, kick
    forces()
    E = [_energy(ctx, vel, inv_m, force, q, alpha)]
    for n in range(NSTEPS):
        ctx.rbe_nve_kick(vel, inv_m, force, 0.5 * DT, pos, xyzq, DT)
        forces()
        ctx.rbe_nve_kick(vel, inv_m, force, 0.5 * DT)
        if (n + 1) % 10 == 0:
            E.append(_energy(ctx, vel, inv_m, force, q, alpha))
    xa, va = pos.cpu().numpy(), vel.cpu().numpy()
    assert np.abs(xa - xs[-1]).max() <= 1e-4, np.abs(xa - xs[-1]).max()
    assert np.abs(va - vs[-1]).max() <= 2e-5, np.abs(va - vs[-1]).max()
    assert np.abs(np.array(E) - Es[::10]).max() <= 2e-6 * abs(Es[0])
    assert np.abs(np.array(E) - E[0]).max() <= 1e-4 * abs(E[0])          # and the loop conserves it
    assert np.array_equal(xyzq.cpu().numpy()[:, :3], xa.astype(np.float32))   # the fp32 copy is kept in step

    # (b) the same 100 steps as 100 replays of ONE captured graph: bitwise the explicit calls
    pos2, vel2, inv_m2, xyzq2, force2 = _gpu_state(x, v, q, mass)
    ctx.rbe_step(None, xyzq2, force2, with_energy=True)
    ctx.rbe_short_range(xyzq2, rs, force2, accumulate=True, with_energy=True)
    ctx.rbe_md_capture(pos2, vel2, inv_m2, xyzq2, force2, rs, DT, sampled=False, with_energy=True)
    for n in range(NSTEPS):
        ctx.rbe_graph_launch()
    torch.cuda.synchronize()
    assert torch.equal(pos2, pos) and torch.equal(vel2, vel) and torch.equal(force2, force)

    # a replay leaves the context on the WEIGHTED k-set it was captured with (regression: rbe_graph_launch used to
    # switch the context back to the uniform weights S/P, so an energy evaluated between replays was wrong)
    tmp = torch.empty_like(force2)
    ctx.rbe_step(None, xyzq2, tmp)
    ref = rbe.Rbe(x.shape[0], L, alpha, m.shape[0])
    ref.rbe_set_kvectors(m, w)
    ref.rbe_step(None, xyzq2, tmp)
    assert ctx.rbe_kspace_energy() == ref.rbe_kspace_energy()


@pytest.mark.parametrize("kind,table", [(0, False), (1, True)], ids=["ring-polynomial", "cells-table"])
def test_random_batch_trajectory_with_the_device_sampler_matches_the_oracle(kind, table):
    """Eq. (2.12) forces from a fresh batch of P = 100 wavevectors per step, drawn on the device (bit-exact against
    oracle/sampler.py), inside the captured graph; the oracle loop uses the same batches.  Once with the default
    real-space kernel, once with the tensor-core cell kernel and the tabulated pair term inside the graph."""
    x, v, q, mass, L, alpha, rs = _system()
    P, seed, step0 = 100, 21, 5
    xs, vs, Es = onve.run(x, v, q, mass, L, alpha, rs, DT, NSTEPS,
                          lambda n: osampler.sample_kset(L, alpha, P, seed, step0 + n))
    ctx = rbe.Rbe(x.shape[0], L, alpha, P)
    ctx.rbe_set_pair_kernel(kind)
    ctx.rbe_set_pair_table(table)
    pos, vel, inv_m, xyzq, force = _gpu_state(x, v, q, mass)
    ctx.rbe_sample_kvectors(seed, step0)
    ctx.rbe_step(None, xyzq, force)
    ctx.rbe_short_range(xyzq, rs, force, accumulate=True)
    ctx.rbe_md_capture(pos, vel, inv_m, xyzq, force, rs, DT, sampled=True, seed=seed, first_step=step0 + 1)
    for n in range(NSTEPS):
        ctx.rbe_graph_launch()
    torch.cuda.synchronize()
    assert np.array_equal(ctx.rbe_get_kvectors(), osampler.sample_kset(L, alpha, P, seed, step0 + NSTEPS))
    assert np.abs(pos.cpu().numpy() - xs[-1]).max() <= 1e-4
    assert np.abs(vel.cpu().numpy() - vs[-1]).max() <= 2e-5
    # momentum: sum_i F_i = 0 for every batch and for the short-range part, so sum m v stays at its start value (0)
    P_tot = (torch.from_numpy(mass).cuda()[:, None] * vel).sum(0).cpu().numpy()
    assert np.abs(P_tot).max() <= 1e-5 * float((torch.from_numpy(mass).cuda()[:, None] * vel.abs()).sum())


def test_energy_sums_and_argument_checks():
    x, v, q, mass, L, alpha, rs = _system()
    ctx = rbe.Rbe(x.shape[0], L, alpha, 8)
    pos, vel, inv_m, xyzq, force = _gpu_state(x, v, q, mass)
    force[:, 3] = torch.arange(x.shape[0], dtype=torch.float32, device="cuda") * 0.25
    ke, sw = ctx.rbe_nve_energies(vel, inv_m, force)
    assert abs(ke - 0.5 * (mass[:, None] * v * v).sum()) <= 1e-13 * ke
    assert sw == 0.25 * x.shape[0] * (x.shape[0] - 1) / 2
    assert ctx.rbe_nve_energies(None, None, force)[0] == 0.0
    # frozen atoms (inverse mass 0) are left out of the kinetic energy instead of turning it into NaN (0 / 0)
    inv_f, vel_f = inv_m.clone(), vel.clone()
    inv_f[:5] = 0.0
    vel_f[:3] = 0.0
    ke_f = ctx.rbe_nve_energies(vel_f, inv_f, force)[0]
    assert abs(ke_f - 0.5 * (mass[5:, None] * v[5:] * v[5:]).sum()) <= 1e-13 * ke
    ctx.rbe_nve_kick(vel_f, inv_f, force, 0.5 * DT)
    assert torch.equal(vel_f[:5], torch.cat([torch.zeros_like(vel[:3]), vel[3:5]]))   # and the kick leaves them alone
    with pytest.raises(rbe.RbeError):
        ctx.rbe_md_capture(pos, vel, inv_m, xyzq, force, rs, DT, sampled=False)        # no k-set yet
    with pytest.raises(rbe.RbeError):
        ctx.rbe_md_capture(pos, vel, inv_m, xyzq, force, rs, -1.0, sampled=True, seed=1)


def test_captured_graph_owns_its_short_range_scratch():
    """The MD graph records the address of its short-range scratch.  The binding used to lend it the context's shared
    scratch tensor, which rbe_short_range / rbe_rbl_forces replace by a larger one when they need more bytes: the graph
    then replayed into freed memory.  Now the graph has a tensor of its own: calls that grow the shared scratch between
    replays change nothing, bit for bit."""
    x, v, q, mass, L, alpha, rs = _system()
    P, seed = 64, 3
    results = []
    for disturb in (False, True):
        ctx = rbe.Rbe(x.shape[0], L, alpha, P)
        pos, vel, inv_m, xyzq, force = _gpu_state(x, v, q, mass)
        ctx.rbe_sample_kvectors(seed, 0)
        ctx.rbe_step(None, xyzq, force)
        ctx.rbe_short_range(xyzq, 0.5 * rs, force, accumulate=True)     # a small shared scratch exists before the capture
        force.zero_()
        ctx.rbe_step(None, xyzq, force)
        ctx.rbe_short_range(xyzq, rs, force, accumulate=True)
        ctx.rbe_md_capture(pos, vel, inv_m, xyzq, force, rs, DT, sampled=True, seed=seed, first_step=1)
        graph_ws = ctx._graph_buffers[-1]
        assert graph_ws.data_ptr() != ctx._sr_ws.data_ptr()
        other = torch.empty_like(force)
        for n in range(20):
            ctx.rbe_graph_launch()
            if disturb and n % 5 == 0:
                ctx._sr_ws = None                                        # the shared scratch is dropped and rebuilt ...
                junk = torch.full((1 << 20,), 0xFF, dtype=torch.uint8, device="cuda")   # ... and its memory reused
                ctx.rbe_rbl_forces(xyzq.clone(), 0.5 * rs, rs, 8, seed, n, other)
                del junk
        torch.cuda.synchronize()
        assert ctx._graph_buffers[-1] is graph_ws
        results.append((pos.clone(), vel.clone(), force.clone()))
    for a, b in zip(*results):
        assert torch.equal(a, b)
