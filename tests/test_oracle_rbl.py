"""Pins of the random-batch-list oracle (oracle/rbl.py; Eqs. 2.13-2.16, reading Q20)."""
import numpy as np

import oracle
from oracle import rbl


def _cell(n, L, seed):
    rng = np.random.default_rng(seed)
    a = np.empty((n, 4), dtype=np.float32)
    a[:, :3] = rng.random((n, 3)) * L
    a[:, 3] = np.where(np.arange(n) % 2 == 0, 1.0, -1.0)
    return a


def test_whole_shell_in_the_batch_reproduces_the_deterministic_sum():
    """p >= N_s for every atom: B(i) = S(i), scale 1, so core + shell = Eq. (2.10) truncated at r_s and the
    correction vanishes with it (Newton's third law)."""
    L, alpha, rc, rs = 24.0, 0.09, 4.0, 8.0
    a = _cell(500, L, 1)
    F, Ns, Fc = rbl.rbl_forces(a, L, alpha, rc, rs, p=10_000, seed=3, step=0)
    Fd, _ = oracle.short_range(a, L, alpha, rs)
    assert np.abs(F - Fd).max() <= 1e-12 * np.abs(Fd).max()
    assert np.abs(Fc).max() <= 1e-13 * np.abs(Fd).max()
    # N_s by brute force for a few atoms
    r = a[:, :3].astype(np.float64)
    for i in (0, 17, 499):
        d = r - r[i]
        d -= L * np.rint(d / L)
        dist = np.sqrt((d * d).sum(1))
        assert Ns[i] == ((dist >= rc) & (dist < rs)).sum()


def test_momentum_is_conserved_exactly_and_the_batch_is_a_p_subset():
    L, alpha, rc, rs, p = 24.0, 0.09, 4.0, 8.0, 12
    a = _cell(500, L, 2)
    F, Ns, Fc = rbl.rbl_forces(a, L, alpha, rc, rs, p, seed=5, step=7)
    assert Ns.min() > p                                      # the random branch is exercised for every atom
    assert np.abs(F.sum(0)).max() <= 1e-12 * np.abs(F).sum()
    F0, _, _ = rbl.rbl_forces(a, L, alpha, rc, rs, p, seed=5, step=7, correction=False)
    assert np.allclose(F0 + Fc, F, rtol=0, atol=1e-15) and np.abs(Fc).max() > 0
    # a different step or seed gives a different batch; the same pair of arguments the same one
    F1, _, _ = rbl.rbl_forces(a, L, alpha, rc, rs, p, seed=5, step=8)
    F2, _, _ = rbl.rbl_forces(a, L, alpha, rc, rs, p, seed=5, step=7)
    assert not np.allclose(F1, F) and np.array_equal(F2, F)
    # keys: a pure function of (seed, step, i, j), uniform on 32 bits
    k = rbl.pair_keys(3, np.arange(20000), 5, 7).astype(np.float64) / 2.0 ** 32
    assert abs(k.mean() - 0.5) < 0.01 and abs(k.var() - 1 / 12) < 0.005
    assert np.array_equal(rbl.pair_keys(3, [11, 12], 5, 7)[1:], rbl.pair_keys(3, [12], 5, 7))
    assert rbl.pair_keys(3, [12], 5, 7)[0] != rbl.pair_keys(12, [3], 5, 7)[0]      # (i, j) is ordered


def test_unbiased_mean_over_steps_converges_to_the_deterministic_force():
    """E[F_i^shell*] = F_i^shell: the residual of the mean over T steps falls like 1/sqrt(T)."""
    L, alpha, rc, rs, p = 18.0, 0.09, 3.0, 7.0, 6
    a = _cell(150, L, 4)
    Fd, _ = oracle.short_range(a, L, alpha, rs)
    acc = np.zeros_like(Fd)
    res = {}
    for t in range(1, 257):
        acc += rbl.rbl_forces(a, L, alpha, rc, rs, p, seed=9, step=t, correction=False)[0]
        if t in (16, 64, 256):
            res[t] = np.linalg.norm(acc / t - Fd)
    assert 1.5 <= res[16] / res[64] <= 2.7 and 1.5 <= res[64] / res[256] <= 2.7, res
    one = np.linalg.norm(rbl.rbl_forces(a, L, alpha, rc, rs, p, seed=9, step=1, correction=False)[0] - Fd)
    assert res[256] <= 0.15 * one


def _fmix32_inverse(h):
    """Inverse of fmix32 from the mathematics, not from its code: x ^= x >> s is undone by repeating the shift-xor
    until the shift passes 32 bits; a multiplication by an odd constant mod 2^32 by its modular inverse."""
    h = int(h)
    h ^= h >> 16
    h = (h * pow(0xC2B2AE35, -1, 1 << 32)) & 0xFFFFFFFF
    h ^= (h >> 13) ^ (h >> 26)
    h = (h * pow(0x85EBCA6B, -1, 1 << 32)) & 0xFFFFFFFF
    h ^= h >> 16
    return h


def test_pair_key_is_a_bijective_well_mixed_hash():
    rng = np.random.default_rng(3)
    x = rng.integers(0, 1 << 32, 2000, dtype=np.uint64)
    y = rbl.fmix32(x)
    assert all(_fmix32_inverse(v) == int(u) for u, v in zip(x, y))          # a bijection, with exactly these steps
    assert int(rbl.fmix32(np.array([0], dtype=np.uint64))[0]) == 0          # fixed point of shift-xor and multiply
    # avalanche: flipping any single input bit flips half of the output bits on average
    for bit in (0, 7, 15, 16, 24, 31):
        flips = np.bitwise_xor(y, rbl.fmix32(x ^ np.uint64(1 << bit)))
        n = np.array([bin(int(v)).count("1") for v in flips])
        assert 15.0 <= n.mean() <= 17.0, (bit, n.mean())
    # for a fixed i the keys of distinct partners are distinct (j -> u_ij is a bijection), and the salt matters
    k = rbl.pair_keys(5, np.arange(50_000), 9, 4)
    assert np.unique(k).shape[0] == 50_000
    assert not np.array_equal(k[:100], rbl.pair_keys(5, np.arange(100), 9, 5))
    assert not np.array_equal(k[:100], rbl.pair_keys(5, np.arange(100), 10, 4))
    assert rbl.step_salt(9, 4) != rbl.step_salt(9, (1 << 32) + 4)                  # the high word of the step counts


def test_batch_is_a_uniform_p_subset_of_the_shell():
    """Every member of S(i) is chosen with probability p / N_s (chi-square over many steps), whatever its index
    or its position in the list -- a selection that favoured low keys' owners, low j, or near neighbours fails."""
    p, T = 6, 3000
    for i, shell in ((0, np.arange(100, 140)), (77, np.array([3, 4, 5, 6, 1000, 1001, 70_000, 2 ** 20 + 1, 12, 13, 14, 15, 16, 17, 18, 19]))):
        counts = np.zeros(shell.shape[0])
        pairs = np.zeros((shell.shape[0], shell.shape[0]))
        for t in range(T):
            keys = rbl.pair_keys(i, shell, 123, t).astype(np.uint64)
            chosen = np.lexsort((shell, keys))[:p]
            counts[chosen] += 1
            pairs[np.ix_(chosen, chosen)] += 1
        n = shell.shape[0]
        expect = T * p / n
        # marginal counts: hypergeometric-like, variance T q (1 - q) with q = p/n; the counts sum to T p exactly
        # (one linear constraint), so sum z^2 has about n - 1 degrees of freedom
        z = (counts - expect) / np.sqrt(T * (p / n) * (1 - p / n))
        assert (z ** 2).sum() <= 2.2 * n, (z ** 2).sum()
        # pair inclusion: P(j and k both in B) = p (p - 1) / (n (n - 1)) for a uniform subset
        off = pairs[~np.eye(n, dtype=bool)]
        q2 = p * (p - 1) / (n * (n - 1))
        assert abs(off.mean() - T * q2) <= 1e-9 * T          # exact: every batch has p (p - 1) ordered pairs
        assert off.std() <= 1.6 * np.sqrt(T * q2 * (1 - q2)), (off.std(), np.sqrt(T * q2))


def test_batches_are_independent_across_atoms_and_across_steps():
    """Eq. (2.15)'s variance and the unbiasedness of the corrected sum need more than the right marginal
    p / N_s: the batches of different atoms, and of one atom at different steps, must not move together.  With
    salted hash keys only 64 bits of salt change from step to step, so this is checked, not assumed: over T steps the
    inclusion indicators X_t(i, j) = [j in B(i)] of (a) two atoms i != i' looking at the same neighbour j, (b) the
    two directions of one pair, X(i, j) and X(j, i), and (c) the same pair at consecutive steps, are uncorrelated --
    sample correlations behave as N(0, 1/T), so the sum of T r^2 over K such combinations is chi-square with about K
    degrees of freedom.  A key that ignored i (every atom picks the same neighbours), a symmetric key (u_ij = u_ji),
    or a salt that moved only a few key bits per step fails by a wide margin (r = 1 gives T per term)."""
    n_atoms, n_i, p, T = 40, 8, 6, 2000
    X = np.zeros((T, n_i, n_atoms), dtype=np.float64)
    for t in range(T):
        for i in range(n_i):
            shell = np.array([j for j in range(n_atoms) if j != i])
            keys = rbl.pair_keys(i, shell, 2024, t).astype(np.uint64)
            X[t, i, shell[np.lexsort((shell, keys))[:p]]] = 1.0
    q = p / (n_atoms - 1)
    assert abs(X.sum() - T * n_i * p) == 0
    Xc = X - q                              # the exact mean of every indicator that is not structurally zero
    var = q * (1 - q)

    def chi2(a, b):
        """sum over the trailing axes of T r^2, r = sample correlation over the step axis (known mean and variance)"""
        r = (a * b).mean(0) / var
        return float((T * r ** 2).sum()), r.size

    # (a) same neighbour j, two different atoms: j runs over the atoms outside 0 .. n_i - 1 (in every shell)
    tot, dof = 0.0, 0
    for i in range(n_i):
        for k in range(i + 1, n_i):
            c, d = chi2(Xc[:, i, n_i:], Xc[:, k, n_i:])
            tot, dof = tot + c, dof + d
    assert dof == 28 * 32 and tot <= dof + 5 * np.sqrt(2 * dof), (tot, dof)
    assert tot >= dof - 5 * np.sqrt(2 * dof), (tot, dof)          # neither correlated nor suspiciously regular
    # (b) the two directions of a pair
    a = np.stack([X[:, i, k] for i in range(n_i) for k in range(i + 1, n_i)], 1) - q
    b = np.stack([X[:, k, i] for i in range(n_i) for k in range(i + 1, n_i)], 1) - q
    tot, dof = chi2(a, b)
    assert dof == 28 and tot <= dof + 5 * np.sqrt(2 * dof), (tot, dof)
    # (c) consecutive steps, same ordered pair
    tot, dof = chi2(Xc[:-1, :, n_i:], Xc[1:, :, n_i:])
    tot *= (T - 1) / T
    assert dof == n_i * 32 and tot <= dof + 5 * np.sqrt(2 * dof), (tot, dof)
    # and a lag of two steps, in case consecutive salts were related pairwise
    tot, dof = chi2(Xc[:-2, :, n_i:], Xc[2:, :, n_i:])
    assert tot <= dof + 5 * np.sqrt(2 * dof), (tot, dof)
