"""Oracle of the counter-based k-vector sampler -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

What it defines (Algorithm 1 step 1; the distribution is P:129: wavevectors
k = 2 pi m / L, m in Z^3 \\ {0}, drawn with probability ~ exp(-|k|^2 / 4 alpha)).  The paper
draws them with a Metropolis chain whose proposal, burn-in and thinning it does not state
(P:129); reading Q2 takes exact iid draws instead (what the unbiasedness
claim P:133 assumes): the pmf factorises per dimension, each m_d comes from the 1-D discrete
Gaussian by inverse CDF, and the triple (0,0,0) is rejected.  DESIGN.md reading Q17 fixes the
random numbers so that a GPU implementation can be compared bit for bit:

  * candidate j = 0, 1, 2, ... of step t with seed s is (x, y, z) = the first three words of
    Philox4x32-10 (Salmon et al., SC'11) with counter (j mod 2^32, j >> 32, t mod 2^32, t >> 32)
    and key (s mod 2^32, s >> 32);
  * 1-D table: c = pi^2 / (alpha L^2), M = ceil(sqrt(40 ln 2 / c)), p_i = exp(-c (i - M)^2) for
    i = 0 .. 2M summed in ascending i (fp64), T_i = floor(2^32 * (p_0 + .. + p_i) / total) for
    i = 0 .. 2M - 1, clamped to 2^32 - 1 (the last bin takes the rest);
  * m_d = #{ i : T_i <= word_d } - M   (an upper bound search: integer comparisons only);
  * the batch is the first P candidates that are not (0, 0, 0), in order of j.

Plain numpy, written out step by step; shares no code with the CUDA path or the harness
sampler in paper_2407_09315_b200/inputs.py.  Pins: tests/test_oracle_sampler.py (the
Random123 known-answer vectors for Philox4x32-10 in tests/golden/philox4x32_10_kat.txt; the
table against the pmf; the rejection rule by brute force; chi-square and second moment).
"""
from __future__ import annotations

import math

import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = 0x9E3779B9
_W1 = 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def philox4x32_10(counter, key):
    """Philox4x32 with 10 rounds.  counter: uint32 [..., 4], key: (k0, k1) -> uint32 [..., 4]."""
    c = np.asarray(counter, dtype=np.uint64) & _MASK
    c0, c1, c2, c3 = c[..., 0], c[..., 1], c[..., 2], c[..., 3]
    k0, k1 = int(key[0]) & 0xFFFFFFFF, int(key[1]) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _M0 * c0                      # 32 x 32 -> 64 bit products
        p1 = _M1 * c2
        hi0, lo0 = p0 >> _S32, p0 & _MASK
        hi1, lo1 = p1 >> _S32, p1 & _MASK
        c0, c1, c2, c3 = (hi1 ^ c1 ^ np.uint64(k0)), lo1, (hi0 ^ c3 ^ np.uint64(k1)), lo0
        k0 = (k0 + _W0) & 0xFFFFFFFF       # key schedule: Weyl sequence
        k1 = (k1 + _W1) & 0xFFFFFFFF
    return np.stack([c0, c1, c2, c3], axis=-1).astype(np.uint32)


def half_width(L: float, alpha: float) -> int:
    c = math.pi * math.pi / (alpha * L * L)
    return int(math.ceil(math.sqrt(40.0 * math.log(2.0) / c)))


def thresholds(L: float, alpha: float):
    """(M, T): T uint32 [2M], T_i = floor(2^32 * CDF(i)) of the 1-D discrete Gaussian on -M..M."""
    c = math.pi * math.pi / (alpha * L * L)
    M = half_width(L, alpha)
    run, cum = 0.0, []
    for i in range(2 * M + 1):             # ascending, sequential fp64 sum; libm exp
        d = float(i - M)
        run += math.exp(-c * (d * d))
        cum.append(run)
    total = cum[-1]
    # clamp: when the tail bins' mass is below fp64 resolution CDF_i rounds to 1 and the floor is 2^32
    T = np.array([min(4294967295, int(math.floor(4294967296.0 * (s / total)))) for s in cum[:-1]], dtype=np.uint64)
    return M, T.astype(np.uint32)


def candidates(L: float, alpha: float, seed: int, step: int, j0: int, n: int) -> np.ndarray:
    """int32 [n,3]: candidates j0 .. j0+n-1 (zero triples included)."""
    M, T = thresholds(L, alpha)
    j = np.arange(j0, j0 + n, dtype=np.uint64)
    ctr = np.stack([j & _MASK, j >> _S32,
                    np.full(n, step & 0xFFFFFFFF, dtype=np.uint64),
                    np.full(n, (step >> 32) & 0xFFFFFFFF, dtype=np.uint64)], axis=-1)
    words = philox4x32_10(ctr, (seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF))[:, :3]
    idx = np.searchsorted(T, words, side="right")          # #{i : T_i <= word}
    return (idx.astype(np.int64) - M).astype(np.int32)


def sample_kset(L: float, alpha: float, P: int, seed: int, step: int) -> np.ndarray:
    """int32 [P,3]: the first P non-zero candidates of (seed, step), in order."""
    out, j0 = [], 0
    have = 0
    while have < P:
        n = max(64, 2 * (P - have))
        cand = candidates(L, alpha, seed, step, j0, n)
        keep = cand[np.any(cand != 0, axis=1)]
        out.append(keep[: P - have])
        have += out[-1].shape[0]
        j0 += n
    return np.ascontiguousarray(np.concatenate(out, axis=0), dtype=np.int32)
