"""Energy drift of the NVE loop against the batch size P.

    python -m paper_2407_09315_b200.nve_drift [--system plasma|rocksalt] [--cells C] [--steps K] [--dt 0.2]
                                              [--seeds 6] [--P 25 50 100 200 400] [--every E]

The system is integrated with velocity Verlet on the GPU, one CUDA-graph launch per step (rbe_md_capture): the
long-range force is either the deterministic Ewald sum (every grid vector, weights exp(-k^2/4alpha): Eq. 2.11) or
its random batch estimate with P wavevectors drawn on the device every step (Eq. 2.12).  Every `--every` steps the
TRUE energy of the state -- kinetic + short-range + deterministic k-space + self term, Eq. 2.8 -- is evaluated by
a second context, whichever force drove the dynamics.  Prints a markdown table: the energy change relative to the
initial kinetic energy (mean and standard deviation over the batch seeds), and the drift rate from a least-squares
line through E(t), multiplied by P (a random force of variance ~ 1/P heats the system at a rate ~ 1/P).

Systems (inputs.py): `plasma` -- a one-component plasma (like charges, implied background), stable without a
repulsive core, for long horizons; `rocksalt` -- the perturbed NaCl crystal of the parity tests, a saddle point
of the pure Coulomb energy that comes apart after ~30 tau, so only a short horizon means anything.
Everything here runs through the C ABI; no oracle, no CPU arithmetic of the method.
"""
from __future__ import annotations

import argparse

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--system", choices=["plasma", "rocksalt"], default="plasma")
    ap.add_argument("--cells", type=int, default=None)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--every", type=int, default=None)
    ap.add_argument("--dt", type=float, default=0.2)
    ap.add_argument("--seeds", type=int, default=6)
    ap.add_argument("--P", type=int, nargs="+", default=[25, 50, 100, 200, 400])
    ap.add_argument("--rs", type=float, default=10.0)
    args = ap.parse_args()

    import torch
    from . import inputs, rbe

    if args.system == "plasma":
        cells, steps = args.cells or 8, args.steps or 2000
        x, v, q, mass, L = inputs.plasma(cells, seed=11, jitter=0.05, v_rms=0.04)
        name = f"one-component plasma, bcc {cells}^3 cells"
    else:
        cells, steps = args.cells or 6, args.steps or 100
        x, v, q, mass, L = inputs.rocksalt(cells, seed=11, jitter=0.05, v_rms=0.04)
        name = f"rock salt {cells}^3 cells"
    every = args.every or max(1, steps // 20)
    N, rs = x.shape[0], min(args.rs, L / 3.0)
    alpha = (3.4 / rs) ** 2
    mmax = int(np.ceil(np.sqrt(18.4 * 4 * alpha) * L / (2 * np.pi)))
    m_full = inputs.full_kgrid(mmax)
    w_full = np.exp(-(2 * np.pi / L) ** 2 * (m_full.astype(np.float64) ** 2).sum(1) / (4 * alpha))
    self_term = -np.sqrt(alpha / np.pi) * float((q.astype(np.float64) ** 2).sum())

    def det_context():
        c = rbe.Rbe(N, L, alpha, m_full.shape[0])
        c.rbe_set_kvectors(m_full, w_full)
        return c

    meter = det_context()            # evaluates the true energy; never drives the dynamics
    scratch = torch.zeros((N, 4), dtype=torch.float32, device="cuda")

    def state():
        pos = torch.from_numpy(x.copy()).cuda()
        vel = torch.from_numpy(v.copy()).cuda()
        inv_m = torch.from_numpy(1.0 / mass).cuda()
        xyzq = torch.from_numpy(np.concatenate([x.astype(np.float32), q[:, None]], axis=1)).cuda().contiguous()
        force = torch.zeros((N, 4), dtype=torch.float32, device="cuda")
        return pos, vel, inv_m, xyzq, force

    def true_energy(xyzq, vel, inv_m):
        meter.rbe_step(None, xyzq, scratch)
        u_k = meter.rbe_kspace_energy()
        meter.rbe_short_range(xyzq, rs, scratch, accumulate=False, with_energy=True)
        ke, u_s = meter.rbe_nve_energies(vel, inv_m, scratch)
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
        for n in range(1, steps + 1):
            ctx.rbe_graph_launch()
            if n % every == 0:
                out.append((true_energy(xyzq, vel, inv_m)[1] - e0) / ke0)
        ke1 = true_energy(xyzq, vel, inv_m)[0]
        return np.array(out), ke0, e0, ke1

    t = np.arange(0, steps + 1, every) * args.dt

    def slope(d):       # least-squares drift rate of (E - E0)/KE0 per tau
        return float(np.polyfit(t[: len(d)], d, 1)[0])

    print(f"# NVE energy drift vs batch size: {name}, N = {N}, L = {L:.2f} A, r_s = {rs:.2f} A, alpha = {alpha:.4f} A^-2,")
    print(f"# dt = {args.dt} tau, {steps} steps ({steps * args.dt:.0f} tau = {steps * args.dt * 2.68285e-3:.2f} ps), true energy every {every} steps; "
          f"deterministic reference: {m_full.shape[0]} wavevectors (|m_d| <= {mmax}); {args.seeds} batch seeds per P")
    d, ke0, e0, ke1 = run(det_context(), False, 0)
    print(f"# E(0) = {e0:.6f} e^2/A, kinetic energy(0) = {ke0:.6f} e^2/A, kinetic energy(end, deterministic run) = {ke1:.6f}\n")
    print("| long-range force | (E - E0)/KE0 at half time: mean ± sd over seeds | at the end: mean ± sd | drift rate [KE0 / tau] | drift rate × P |")
    print("|---|---|---|---|---|")
    h = len(d) // 2
    print(f"| deterministic Ewald (Eq. 2.11) | {d[h]:+.2e} | {d[-1]:+.2e} | {slope(d):+.2e} | — |")
    for P in args.P:
        ctx = rbe.Rbe(N, L, alpha, P)
        runs = np.array([run(ctx, True, 1000 + s)[0] for s in range(args.seeds)])
        rates = np.array([slope(r) for r in runs])
        print(f"| random batch, P = {P} (Eq. 2.12) | {runs[:, h].mean():+.2e} ± {runs[:, h].std():.1e} | "
              f"{runs[:, -1].mean():+.2e} ± {runs[:, -1].std():.1e} | {rates.mean():+.2e} ± {rates.std():.1e} | {rates.mean() * P:+.2e} |")


if __name__ == "__main__":
    main()
