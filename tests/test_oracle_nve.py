"""Pins of the NVE velocity-Verlet oracle (oracle/nve.py; PAPER.md P:78 velocity-Verlet, P:86 NVE)."""
import numpy as np

import oracle
from oracle import nve
from paper_2407_09315_b200 import inputs


def _system(ncells=2, jitter=0.05, v_rms=0.04, seed=7):
    x, v, q, mass, L = inputs.rocksalt(ncells, seed=seed, jitter=jitter, v_rms=v_rms)
    rs = L / 3.0
    alpha = (3.4 / rs) ** 2                      # erfc(sqrt(alpha) r_s) = 1.5e-6: the truncated tail is negligible
    mmax = int(np.ceil(np.sqrt(18.4 * 4 * alpha) * L / (2 * np.pi)))     # exp(-k^2/4alpha) < 1e-8 beyond it
    m = inputs.full_kgrid(mmax)
    w = np.exp(-(2 * np.pi / L) ** 2 * (m.astype(np.float64) ** 2).sum(1) / (4 * alpha))
    return x, v, q, mass, L, alpha, rs, m, w


def test_potential_energy_is_the_ewald_energy_and_the_force_its_gradient():
    """total_force's energy = the three terms of Eq. (2.8) as oracle.ewald_full sums them (real-space images, full
    k-grid, self), up to the pairs beyond r_s; its force is minus the gradient of ITS energy (central differences),
    which is what makes the energy of the loop a conserved quantity."""
    x, v, q, mass, L, alpha, rs, m, w = _system()
    x32 = x.astype(np.float32).astype(np.float64)
    F, U = nve.total_force(x32, q, L, alpha, rs, m, w)
    Uref, Fs, Fl = oracle.ewald_full(x32, q.astype(np.float64), L, alpha, nreal=2, mmax=int(np.abs(m).max()))
    assert abs(U - Uref.sum()) <= 1e-5 * abs(Uref.sum())          # the tail beyond r_s: erfc(3.4)/r per pair
    assert np.linalg.norm(F - (Fs + Fl)) <= 1e-4 * np.linalg.norm(Fs + Fl)
    h = 2e-3                                                      # positions are rounded to fp32 inside: keep h >> 1e-6
    for i, d in ((0, 0), (5, 2), (60, 1)):
        xp, xm = x32.copy(), x32.copy()
        xp[i, d] += h; xm[i, d] -= h
        xp, xm = xp.astype(np.float32).astype(np.float64), xm.astype(np.float32).astype(np.float64)
        g = (nve.total_force(xp, q, L, alpha, rs, m, w)[1] - nve.total_force(xm, q, L, alpha, rs, m, w)[1]) / (xp[i, d] - xm[i, d])
        assert abs(-g - F[i, d]) <= 2e-4 * np.abs(F).max(), (i, d, -g, F[i, d])


def test_first_step_from_rest_and_momentum():
    """From rest, x(dt) = x(0) + dt^2 F(0) / (2 m) and v(dt) = dt (F(0) + F(dt)) / (2 m): the scheme of the docstring
    checked against forces evaluated separately; total momentum stays zero to rounding."""
    x, v, q, mass, L, alpha, rs, m, w = _system(v_rms=0.0)
    dt = 0.25
    xs, vs, Es = nve.run(x, v, q, mass, L, alpha, rs, dt, 3, m, w)
    F0, _ = nve.total_force(x, q, L, alpha, rs, m, w)
    assert np.allclose(xs[1], x + dt * dt * F0 / (2 * mass[:, None]), rtol=0, atol=1e-14)
    F1, _ = nve.total_force(xs[1], q, L, alpha, rs, m, w)
    assert np.allclose(vs[1], dt * (F0 + F1) / (2 * mass[:, None]), rtol=0, atol=1e-15)
    P = (mass[None, :, None] * vs).sum(1)
    assert np.abs(P).max() <= 1e-12 * np.abs(mass[None, :, None] * vs).sum(1).max()


def test_time_reversible():
    x, v, q, mass, L, alpha, rs, m, w = _system()
    xs, vs, _ = nve.run(x, v, q, mass, L, alpha, rs, 0.2, 20, m, w)
    xb, vb, _ = nve.run(xs[-1], -vs[-1], q, mass, L, alpha, rs, 0.2, 20, m, w)
    # exact in real arithmetic; in fp64 with forces taken on fp32-rounded positions the return error is a few ulp(fp32)
    assert np.abs(xb[-1] - x).max() <= 2e-5 and np.abs(vb[-1] + v).max() <= 2e-5
    assert np.abs(xs[10] - xb[10]).max() <= 2e-5


def test_energy_error_is_second_order_in_dt():
    """Deterministic mode (weighted full k-grid): max |E(t) - E(0)| over the same time span falls ~4 x when dt is
    halved, down to the floor set by evaluating the forces on fp32-rounded positions (~1e-5 e^2/A here)."""
    x, v, q, mass, L, alpha, rs, m, w = _system()
    span = 16.0
    err = {}
    for dt in (1.6, 0.8, 0.4):
        _, _, E = nve.run(x, v, q, mass, L, alpha, rs, dt, int(round(span / dt)), m, w)
        err[dt] = np.abs(E - E[0]).max()
    assert 3.0 <= err[1.6] / err[0.8] <= 5.0 and 3.0 <= err[0.8] / err[0.4] <= 5.0, err
    assert err[0.4] <= 1e-5 * abs(E[0])


def test_random_batch_forces_replace_the_long_range_part():
    """kset as a callable: evaluation n uses its own batch; with one batch repeated the loop equals the fixed-set loop."""
    x, v, q, mass, L, alpha, rs, m, w = _system()
    batch = inputs.sample_kset(L, alpha, 50, 3, 0)
    a = nve.run(x, v, q, mass, L, alpha, rs, 0.2, 4, batch)
    b = nve.run(x, v, q, mass, L, alpha, rs, 0.2, 4, lambda n: batch)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[2], b[2])
    c = nve.run(x, v, q, mass, L, alpha, rs, 0.2, 4, lambda n: inputs.sample_kset(L, alpha, 50, 3, n))
    assert not np.array_equal(a[0][-1], c[0][-1])
