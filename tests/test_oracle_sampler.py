"""Pins of the counter-based k-vector sampler oracle (oracle/sampler.py, reading Q17):
Algorithm 1 step 1, distribution of P:129."""
import os

import numpy as np

from oracle import sampler
from paper_2407_09315_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers():
    rows = [l.split() for l in open(GOLDEN) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = sampler.philox4x32_10(np.array(v[:4]), (v[4], v[5]))
        assert [int(x) for x in out] == v[6:]
    # vectorised call = element-wise calls
    ctr = np.array([[1, 2, 3, 4], [5, 6, 7, 8]])
    both = sampler.philox4x32_10(ctr, (9, 10))
    assert np.array_equal(both[1], sampler.philox4x32_10(ctr[1], (9, 10)))


def test_thresholds_reproduce_the_pmf():
    for L, alpha in [(31.04, 0.09), (215.443, 0.09), (12.0, 0.3), (1000.0, 0.09)]:
        M, T = sampler.thresholds(L, alpha)
        assert T.shape == (2 * M,) and np.all(np.diff(T.astype(np.int64)) >= 0)
        # bin masses from the integer thresholds against the closed-form pmf (harness, independent code)
        edges = np.concatenate([[0], T.astype(np.float64), [2.0 ** 32]])
        mass = np.diff(edges) / 2.0 ** 32
        ms, p = inputs.pmf_1d(L, alpha)
        ref = dict(zip(ms.tolist(), p.tolist()))
        for i, m in enumerate(range(-M, M + 1)):
            assert abs(mass[i] - ref.get(m, 0.0)) <= 2.0 ** -31
        # symmetric to within one count, and the tail beyond M is below the 2^-32 resolution
        assert np.abs(mass - mass[::-1]).max() <= 2.0 ** -31
        c = np.pi ** 2 / (alpha * L * L)
        assert np.exp(-c * (M + 1) ** 2) < 2.0 ** -40


def test_rejection_rule_by_brute_force():
    """Small box: zero triples are frequent; the batch is the first P non-zero candidates in order."""
    L, alpha, P = 6.0, 0.3, 200
    cand = sampler.candidates(L, alpha, seed=7, step=3, j0=0, n=4000)
    nz = [tuple(c) for c in cand.tolist() if any(c)]
    assert len(nz) < 4000 * 0.95          # the rule is exercised
    got = sampler.sample_kset(L, alpha, P, 7, 3)
    assert [tuple(x) for x in got.tolist()] == nz[:P]
    assert np.all(np.any(got != 0, axis=1))
    # candidates are a pure function of (seed, step, j): windows agree, steps and seeds differ
    assert np.array_equal(sampler.candidates(L, alpha, 7, 3, 100, 50), cand[100:150])
    assert not np.array_equal(sampler.candidates(L, alpha, 7, 4, 0, 50), cand[:50])
    assert not np.array_equal(sampler.candidates(L, alpha, 8, 3, 0, 50), cand[:50])
    big = sampler.candidates(L, alpha, 7, (1 << 40) + 3, 0, 50)   # high word of the step is used
    assert not np.array_equal(big, cand[:50])


def test_distribution_chi_square_and_second_moment():
    L, alpha = 31.04, 0.09
    m = sampler.sample_kset(L, alpha, 200_000, seed=11, step=0)
    ms, p = inputs.pmf_1d(L, alpha)
    # conditional on m != 0 the per-dimension marginal is p(m) (1 - [m=0] p0^2) / (1 - p0^3)
    p0 = float(p[ms == 0][0])
    marg = p * np.where(ms == 0, 1 - p0 ** 2, 1.0) / (1 - p0 ** 3)
    keep = marg * m.shape[0] >= 20
    for d in range(3):
        cnt = np.array([(m[:, d] == v).sum() for v in ms[keep]])
        exp = marg[keep] * m.shape[0]
        chi2 = ((cnt - exp) ** 2 / exp).sum()
        dof = keep.sum() - 1
        assert chi2 < dof + 6 * np.sqrt(2 * dof), (d, chi2, dof)
    # E[m_d^2] ~ alpha L^2 / (2 pi^2) (continuum variance), corrected for the rejected origin
    var = (marg * ms.astype(np.float64) ** 2).sum()
    assert abs((m.astype(np.float64) ** 2).mean() - var) < 0.02 * var
    assert abs(var - alpha * L * L / (2 * np.pi ** 2)) < 0.02 * var


def test_same_law_as_the_harness_sampler():
    """Two independent implementations of reading Q2 (this one: Philox + integer thresholds; the
    harness: PCG64 + float CDF) agree in distribution: compare |m|^2 histograms."""
    L, alpha, n = 98.65, 0.09, 100_000
    a = (sampler.sample_kset(L, alpha, n, 5, 0).astype(np.int64) ** 2).sum(1)
    b = (inputs.sample_kset(L, alpha, n, 5, 0).astype(np.int64) ** 2).sum(1)
    edges = np.quantile(np.concatenate([a, b]), np.linspace(0, 1, 21))
    ha, _ = np.histogram(a, edges)
    hb, _ = np.histogram(b, edges)
    chi2 = ((ha - hb) ** 2 / np.maximum(ha + hb, 1)).sum()
    assert chi2 < 19 + 6 * np.sqrt(38), chi2
