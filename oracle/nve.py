"""Oracle of the NVE velocity-Verlet loop -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md: "All these forces are summed up and assigned to each atom for the velocity-Verlet time
integration"; the NVE ensemble is among those the package runs; the paper's outlook asks how
the random batch forces behave in long runs.  SURVEY.md s8(f) row 4 asks for a minimal NVE loop that
shows the energy drift against the batch size P.

The velocity-Verlet scheme written out (fp64, plain numpy, one step at a time), for point charges with masses
m_i moving under F_i = F_i^short (Eq. 2.10, truncated at r_s, oracle.short_range) + F_i^long
(Eq. 2.11 P:125 over a weighted k-set, or its random batch estimate Eq. 2.12, oracle.force):

    v(t + dt/2) = v(t) + (dt / 2) F(x(t)) / m
    x(t + dt)   = x(t) + dt v(t + dt/2)
    v(t + dt)   = v(t + dt/2) + (dt / 2) F(x(t + dt)) / m

Units (reading Q21): Gaussian as everywhere on this path -- lengths in A, charges in e, forces in
e^2/A^2, energies in e^2/A -- masses in amu, hence times in tau = sqrt(amu A^3 / e^2) = 2.6829 fs.

The forces are evaluated on the positions ROUNDED TO fp32, as the GPU path sees them (its kernels take float4
{x, y, z, q}); the state (x, v) itself stays fp64 on both sides.  Nothing keeps unlike charges apart on this
path (the paper's Lennard-Jones term, Eq. 2.2, is out of scope): the loop is meant for SHORT horizons from a
perturbed rock-salt lattice, where every ion stays near its site.

Pins (tests/test_oracle_nve.py): time reversibility (forward n steps, negate v, n steps back: the start to
rounding); conservation of total momentum to rounding (sum_i F_i = 0 for both parts of the force); the energy
error of the deterministic mode falls 4 x when dt is halved (second order) with the energy taken from
oracle.ewald_full's terms; one step against the three formulas above retyped for a single particle pair in a
closed form (two charges on the x axis, first step from rest: x_1(dt) = x_1(0) + dt^2 F / (2 m)).
"""
from __future__ import annotations

import math

import numpy as np

from . import S as _S, energy as _energy, force as _force, rho as _rho, short_range as _short_range

TAU_FS = 2.68285  # sqrt(amu A^3 / e^2) in femtoseconds (context only; nothing below uses it)


def total_force(x, q, L, alpha, rs, m, w=None):
    """F_short + F_long and the potential energy (short + k-space + self) at positions x (fp64 [N,3]).

    w = None: random batch weights S / P for the k-set m (Eq. 2.12); else the given weights (w_l =
    exp(-k_l^2 / 4 alpha) over the full grid = Eq. 2.11)."""
    xyzq = np.empty((x.shape[0], 4), dtype=np.float32)
    xyzq[:, :3] = x                                          # the rounding the GPU path sees
    xyzq[:, 3] = q
    Fs, es = _short_range(xyzq, L, alpha, rs)
    S = _S(L, alpha)
    rho = _rho(xyzq, L, m)
    Fl = _force(xyzq, L, m, S, rho, w=w)
    U = float(es.sum()) + _energy(L, m, S, rho, w=w) - math.sqrt(alpha / math.pi) * float((q.astype(np.float64) ** 2).sum())
    return Fs + Fl, U


def run(x0, v0, q, mass, L, alpha, rs, dt, nsteps, kset, w=None):
    """Velocity Verlet for nsteps.  kset: int32 [P,3] (one fixed set, e.g. the full grid with weights w) or a
    callable step -> int32 [P,3] (a fresh random batch per force evaluation; evaluation n uses kset(n), the
    initial forces are evaluation 0).  Returns (x [nsteps+1,N,3], v [nsteps+1,N,3], E [nsteps+1] = kinetic +
    potential with the SAME k-set the forces of that time used)."""
    x = np.array(x0, dtype=np.float64)
    v = np.array(v0, dtype=np.float64)
    q = np.asarray(q, dtype=np.float32)
    inv_m = 1.0 / np.asarray(mass, dtype=np.float64)[:, None]
    ks = kset if callable(kset) else (lambda n: kset)
    F, U = total_force(x, q, L, alpha, rs, ks(0), w)
    xs, vs, Es = [x.copy()], [v.copy()], [0.5 * float((v * v / inv_m).sum()) + U]
    for n in range(1, nsteps + 1):
        v = v + (0.5 * dt) * F * inv_m
        x = x + dt * v
        F, U = total_force(x, q, L, alpha, rs, ks(n), w)
        v = v + (0.5 * dt) * F * inv_m
        xs.append(x.copy()); vs.append(v.copy()); Es.append(0.5 * float((v * v / inv_m).sum()) + U)
    return np.array(xs), np.array(vs), np.array(Es)
