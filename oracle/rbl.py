"""Oracle of the random batch list (RBL) short-range force -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md section 2.3, Eqs. (2.13)-(2.16) and Algorithm 2, applied to the only
short-range pair force this path has, the electrostatic one of Eq. (2.10) P:122:

  C(i) = { j != i : r_ij < r_c },   S(i) = { j : r_c <= r_ij < r_s }                       Eq. (2.13)
  F_i^core  = sum_{j in C(i)} F_ij            (direct sum)                                   Eq. (2.14)
  F_i^shell* = (N_s / p) sum_{j in B(i)} F_ij,   B(i) = p random members of S(i), N_s = |S(i)|   Eq. (2.15)
  F^corr = -(1 / N) sum_i (F_i^core + F_i^shell*)                                            Eq. (2.16)
  F_i = F_i^core + F_i^shell* + F^corr

  F_ij = - q_i q_j ( erfc(sqrt(alpha) r)/r^2 + 2 sqrt(alpha) exp(-alpha r^2)/(sqrt(pi) r) ) d / r,
  d = nearest image of r_j - r_i, r = |d|                                                     Eq. (2.10)

DESIGN.md reading Q20 (the paper says "randomly chooses a few p particles from S(i)", and gives
no procedure): every shell pair gets a 32-bit key u_ij and B(i) is the set of the min(p, N_s) members of
S(i) with the smallest (u_ij, j).  The key is a salted integer hash of the ordered pair (i, j = atom indices):

  (s0, s1) = first two words of Philox4x32-10 with counter (step mod 2^32, step >> 32, 0, 0) and key
             (seed mod 2^32, seed >> 32)                                  -- one call per step, not per pair
  u_ij     = fmix32( (i * 0x9E3779B1 + s0) xor (j * 0x85EBCA77 + s1) )    -- all arithmetic mod 2^32
  fmix32(h): h ^= h >> 16; h *= 0x85EBCA6B; h ^= h >> 13; h *= 0xC2B2AE35; h ^= h >> 16
             (the 32-bit finaliser of Appleby's MurmurHash3, public domain: a bijection with full avalanche)

For a fixed i the map j -> u_ij is a bijection of the 32-bit integers (odd multiplier, xor with a constant,
bijective finaliser), so the keys of a shell are distinct, the p smallest are well defined, and -- the salt
being fresh every step -- B(i) behaves as a uniformly random p-subset of S(i) (without replacement),
independent of the order in which an implementation meets the neighbours, and a GPU implementation can
reproduce it exactly.  (Round 1 used one Philox4x32-10 call per shell pair: statistically the same batch law
at six times the integer work per pair; revised so that choosing the batch costs less than evaluating the
shell it replaces, which is the point of P:154-166.)  If N_s <= p the whole shell is summed (scale 1).  The
outer cutoff is strict (r < r_s, reading Q18).

Plain numpy, fp64, one atom at a time: O(N^2).  Pins (tests/test_oracle_rbl.py): p >= max N_s
reproduces oracle.short_range exactly; sum_i F_i = 0 after the correction; the mean over steps
converges to oracle.short_range (unbiasedness) with the 1/sqrt(T) law; the keys: bijectivity of
fmix32 (inverted with the modular inverses of its multipliers), avalanche, and a chi-square test that every
shell member is picked with probability p / N_s, and correlation tests that the batches of different atoms, of the two
directions of a pair and of consecutive steps are independent; Philox itself by the Random123 vectors
(tests/test_oracle_sampler.py).
"""
from __future__ import annotations

import math

import numpy as np

from .sampler import philox4x32_10


_M32 = np.uint64(0xFFFFFFFF)


def fmix32(h) -> np.ndarray:
    """The MurmurHash3 32-bit finaliser on an array of uint32 (computed in uint64, reduced mod 2^32)."""
    h = np.asarray(h, dtype=np.uint64) & _M32
    h ^= h >> np.uint64(16)
    h = (h * np.uint64(0x85EBCA6B)) & _M32
    h ^= h >> np.uint64(13)
    h = (h * np.uint64(0xC2B2AE35)) & _M32
    h ^= h >> np.uint64(16)
    return h.astype(np.uint32)


def step_salt(seed: int, step: int):
    """(s0, s1): the per-step salt, one Philox4x32-10 call."""
    w = philox4x32_10(np.array([[step & 0xFFFFFFFF, (step >> 32) & 0xFFFFFFFF, 0, 0]], dtype=np.uint64),
                      (seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF))[0]
    return int(w[0]), int(w[1])


def pair_keys(i: int, js, seed: int, step: int) -> np.ndarray:
    """uint32 keys u_ij for the atom i and the array of partner indices js."""
    s0, s1 = step_salt(seed, step)
    js = np.asarray(js, dtype=np.uint64)
    a = np.uint64((int(i) * 0x9E3779B1 + s0) & 0xFFFFFFFF)
    b = (js * np.uint64(0x85EBCA77) + np.uint64(s1)) & _M32
    return fmix32(a ^ b)


def rbl_forces(xyzq, L: float, alpha: float, rc: float, rs: float, p: int, seed: int, step: int,
               sel=None, correction: bool = True):
    """Returns (F float64 [nsel,3], Ns int64 [nsel], Fcorr float64 [3]).  With `sel` the correction still
    needs every atom, so all atoms are evaluated and the selected rows returned."""
    a = np.ascontiguousarray(xyzq, dtype=np.float32).astype(np.float64)
    N = a.shape[0]
    assert 0 < rc < rs <= 0.5 * L + 1e-12
    r, q = a[:, :3], a[:, 3]
    sa = math.sqrt(alpha)
    erfc = np.vectorize(math.erfc, otypes=[np.float64])
    F = np.zeros((N, 3))
    Ns = np.zeros(N, dtype=np.int64)
    for i in range(N):
        d = r - r[i]
        d -= L * np.rint(d / L)                                     # nearest image
        dist = np.sqrt((d * d).sum(1))
        core = np.nonzero((dist < rc) & (dist > 0.0))[0]
        shell = np.nonzero((dist >= rc) & (dist < rs))[0]
        Ns[i] = shell.shape[0]
        if shell.shape[0] > p:
            keys = pair_keys(i, shell, seed, step).astype(np.uint64)
            order = np.lexsort((shell, keys))                        # by key, ties by j
            batch, scale = shell[order[:p]], shell.shape[0] / p
        else:
            batch, scale = shell, 1.0
        for idx, w in ((core, 1.0), (batch, scale)):
            if idx.shape[0] == 0:
                continue
            rr = dist[idx]
            g = erfc(sa * rr) / rr ** 2 + 2.0 * sa * np.exp(-alpha * rr ** 2) / (math.sqrt(math.pi) * rr)
            F[i] += w * (-(q[i] * q[idx] * g / rr)[:, None] * d[idx]).sum(0)
    Fcorr = -F.sum(0) / N if correction else np.zeros(3)
    F = F + Fcorr
    if sel is not None:
        sel = np.asarray(sel, dtype=np.int64)
        return F[sel], Ns[sel], Fcorr
    return F, Ns, Fcorr
