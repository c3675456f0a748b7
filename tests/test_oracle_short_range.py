"""Pins of the short-range oracle (oracle/short_range.c): Eq. (2.10) P:122 truncated at r_s."""
import math

import numpy as np

import oracle


def _cell(n, L, seed):
    rng = np.random.default_rng(seed)
    a = np.empty((n, 4), dtype=np.float32)
    a[:, :3] = rng.random((n, 3)) * L
    a[:, 3] = np.where(np.arange(n) % 2 == 0, 1.0, -1.0) * (0.5 + rng.random(n))
    return a


def test_matches_the_full_ewald_real_space_sum_when_the_cutoff_is_harmless():
    """alpha r_s^2 = 36: erfc(6) = 2e-17, so truncation at r_s = L/2 changes nothing and the result
    must equal oracle.ewald_full's real-space part (pinned by the Madelung constant) with images."""
    L, alpha = 12.0, 1.0
    a = _cell(40, L, 1)
    F, e = oracle.short_range(a, L, alpha, rs=L / 2)
    U, Fs, _ = oracle.ewald_full(a[:, :3].astype(np.float64), a[:, 3].astype(np.float64), L, alpha, nreal=1, mmax=0)
    assert np.abs(F - Fs).max() <= 1e-13 * np.abs(Fs).max()
    assert abs(e.sum() - U[0]) <= 1e-13 * abs(U[0])


def test_two_charges_closed_form_and_direction():
    L, alpha, rs = 20.0, 0.09, 9.0
    q1, q2, d = 0.7, 1.3, 3.0
    a = np.array([[19.0, 5.0, 5.0, q1], [19.0 + d - L, 5.0, 5.0, q2]], dtype=np.float32)   # across the boundary
    F, e = oracle.short_range(a, L, alpha, rs)
    q1, q2 = float(a[0, 3]), float(a[1, 3])      # the fp32 charges the oracle sees
    sa = math.sqrt(alpha)
    g = math.erfc(sa * d) / d ** 2 + 2 * sa * math.exp(-alpha * d * d) / (math.sqrt(math.pi) * d)
    assert np.allclose(F[0], [-q1 * q2 * g, 0, 0], rtol=1e-12, atol=1e-15)   # like charges repel: pushed to -x
    assert np.allclose(F[1], [+q1 * q2 * g, 0, 0], rtol=1e-12, atol=1e-15)
    assert np.allclose(e, 0.5 * q1 * q2 * math.erfc(sa * d) / d, rtol=1e-12)
    # beyond the cutoff: nothing
    a[1, 0] = np.float32(19.0 + 9.5 - L)
    F, e = oracle.short_range(a, L, alpha, rs)
    assert np.all(F == 0.0) and np.all(e == 0.0)


def test_newton_third_law_and_cutoff_rule_by_brute_force():
    L, alpha, rs = 30.0, 0.09, 8.0
    a = _cell(300, L, 2)
    F, e = oracle.short_range(a, L, alpha, rs)
    assert np.abs(F.sum(0)).max() <= 1e-12 * np.abs(F).sum()
    # independent brute force in numpy over explicit images
    r = a[:, :3].astype(np.float64)
    q = a[:, 3].astype(np.float64)
    Fb = np.zeros_like(r)
    sa = math.sqrt(alpha)
    for n in np.ndindex(3, 3, 3):
        d = r[None, :, :] - r[:, None, :] + (np.array(n) - 1) * L          # d[i,j] = r_j - r_i + nL
        dist = np.sqrt((d ** 2).sum(-1))
        mask = (dist < rs) & (dist > 0)
        dd = np.where(mask, dist, 1.0)
        g = np.vectorize(math.erfc)(sa * dd) / dd ** 2 + 2 * sa * np.exp(-alpha * dd ** 2) / (math.sqrt(math.pi) * dd)
        Fb += (-(q[:, None] * q[None, :] * g * mask)[:, :, None] * d / dd[:, :, None]).sum(1)
    assert np.abs(F - Fb).max() <= 1e-12 * np.abs(Fb).max()
    # sel = subset gives the same rows
    sel = np.array([5, 17, 299], dtype=np.int64)
    Fs, es = oracle.short_range(a, L, alpha, rs, sel=sel)
    assert np.array_equal(Fs, F[sel]) and np.array_equal(es, e[sel])


def test_force_is_minus_gradient_of_the_energy_away_from_the_cutoff():
    L, alpha = 12.0, 1.0                       # cutoff harmless (see first test): U is smooth
    a = _cell(12, L, 3)
    F, e = oracle.short_range(a, L, alpha, rs=L / 2)
    h = 2.0 ** -10                             # exactly representable steps in fp32 coordinates
    for i, d in ((0, 0), (5, 1), (11, 2)):
        ap, am = a.copy(), a.copy()
        ap[i, d] += np.float32(h)
        am[i, d] -= np.float32(h)
        step = float(ap[i, d]) - float(am[i, d])
        dU = (oracle.short_range(ap, L, alpha, L / 2)[1].sum() - oracle.short_range(am, L, alpha, L / 2)[1].sum()) / step
        assert abs(-dU - F[i, d]) <= 1e-5 * np.abs(F).max()
