"""Energy drift of the NVE loop against the batch size P.

    python -m paper_2407_09315_b200.nve_drift [--cells 6] [--steps 100] [--dt 0.2] [--seeds 6] [--P 50 100 200 400]

A perturbed rock-salt crystal (inputs.rocksalt) is integrated with velocity Verlet on the GPU, one CUDA-graph
launch per step (rbe_md_capture): the long-range force is either the deterministic Ewald sum (every grid vector,
weights exp(-k^2/4alpha): Eq. 2.11) or its random batch estimate with P wavevectors drawn on the device every step
(Eq. 2.12).  Every 10 steps the TRUE energy of the state -- kinetic + short-range + deterministic k-space + self
term, Eq. 2.8 -- is evaluated, whichever force drove the dynamics.  Prints a markdown table: the energy change
relative to the initial kinetic energy, mean and root mean square over the batch seeds.

The horizon is short on purpose: this path has no repulsive core (the paper's Lennard-Jones term is out of scope),
and a pure Coulomb crystal is a saddle point -- it comes apart after ~30 tau.
Everything here runs through the C ABI; no oracle, no CPU arithmetic of the method.
"""
from __future__ import annotations

import argparse

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cells", type=int, default=6)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--dt", type=float, default=0.2)
    ap.add_argument("--seeds", type=int, default=6)
    ap.add_argument("--P", type=int, nargs="+", default=[50, 100, 200, 400])
    ap.add_argument("--rs", type=float, default=10.0)
    args = ap.parse_args()

    import torch
    from . import inputs, rbe

    x, v, q, mass, L = inputs.rocksalt(args.cells, seed=11, jitter=0.05, v_rms=0.04)
    N, rs = x.shape[0], min(args.rs, L / 3.0)
    alpha = (3.4 / rs) ** 2
    mmax = int(np.ceil(np.sqrt(18.4 * 4 * alpha) * L / (2 * np.pi)))
    m_full = inputs.full_kgrid(mmax)
    w_full = np.exp(-(2 * np.pi / L) ** 2 * (m_full.astype(np.float64) ** 2).sum(1) / (4 * alpha))
    self_term = -np.sqrt(alpha / np.pi) * float((q.astype(np.float64) ** 2).sum())

    det = rbe.Rbe(N, L, alpha, m_full.shape[0])
    det.rbe_set_kvectors(m_full, w_full)
    scratch = torch.zeros((N, 4), dtype=torch.float32, device="cuda")

    def state():
        pos = torch.from_numpy(x.copy()).cuda()
        vel = torch.from_numpy(v.copy()).cuda()
        inv_m = torch.from_numpy(1.0 / mass).cuda()
        xyzq = torch.from_numpy(np.concatenate([x.astype(np.float32), q[:, None]], axis=1)).cuda().contiguous()
        force = torch.zeros((N, 4), dtype=torch.float32, device="cuda")
        return pos, vel, inv_m, xyzq, force

    def true_energy(xyzq, vel, inv_m):
        det.rbe_step(None, xyzq, scratch)
        u_k = det.rbe_kspace_energy()
        det.rbe_short_range(xyzq, rs, scratch, accumulate=False, with_energy=True)
        ke, u_s = det.rbe_nve_energies(vel, inv_m, scratch)
        return ke, ke + u_s + u_k + self_term

    def run(ctx, sampled, seed):
        pos, vel, inv_m, xyzq, force = state()
        if sampled:
            ctx.rbe_sample_kvectors(seed, 0)
        ctx.rbe_step(None, xyzq, force)
        ctx.rbe_short_range(xyzq, rs, force, accumulate=True)
        ctx.rbe_md_capture(pos, vel, inv_m, xyzq, force, rs, args.dt, sampled=sampled, seed=seed, first_step=1)
        ke0, e0 = true_energy(xyzq, vel, inv_m)
        out = [0.0]
        for n in range(1, args.steps + 1):
            ctx.rbe_graph_launch()
            if n % 10 == 0:
                out.append((true_energy(xyzq, vel, inv_m)[1] - e0) / ke0)
        return np.array(out), ke0, e0

    print(f"# NVE energy drift vs batch size: rock salt {args.cells}^3 cells, N = {N}, L = {L:.2f} A, r_s = {rs:.2f} A, alpha = {alpha:.4f} A^-2,")
    print(f"# dt = {args.dt} tau, {args.steps} steps ({args.steps * args.dt:.0f} tau = {args.steps * args.dt * 2.68285:.0f} fs), deterministic reference: "
          f"{m_full.shape[0]} wavevectors (|m_d| <= {mmax}); {args.seeds} batch seeds per P")
    d, ke0, e0 = run(det, False, 0)
    print(f"# E(0) = {e0:.6f} e^2/A, kinetic energy(0) = {ke0:.6f} e^2/A\n")
    print("| long-range force | (E - E0)/KE0 at 50 % of the run: mean, rms over seeds | at the end: mean, rms | max |E - E0|/KE0 over the run |")
    print("|---|---|---|---|")
    h = len(d) // 2
    print(f"| deterministic Ewald (Eq. 2.11) | {d[h]:+.2e} | {d[-1]:+.2e} | {np.abs(d).max():.2e} |")
    for P in args.P:
        ctx = rbe.Rbe(N, L, alpha, P)
        runs = np.array([run(ctx, True, 1000 + s)[0] for s in range(args.seeds)])
        print(f"| random batch, P = {P} (Eq. 2.12) | {runs[:, h].mean():+.2e}, {np.sqrt((runs[:, h] ** 2).mean()):.2e} | "
              f"{runs[:, -1].mean():+.2e}, {np.sqrt((runs[:, -1] ** 2).mean()):.2e} | {np.abs(runs).max():.2e} |")


if __name__ == "__main__":
    main()
