"""Oracle of the k-space virial -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The paper names the isothermal-isobaric variant of the RBE without giving the pressure
estimator; reading Q19 takes the strain derivative of the second term of Eq. (2.8)
with the same importance weights as the force (Eq. 2.12) and the energy (reading Q7).  Under a
homogeneous strain eps (r -> (1 + eps) r, box likewise) k . r and therefore rho(k) are invariant,
V -> V (1 + tr eps), k^2 -> k^2 - 2 k_a k_b eps_ab, so with g(k) = exp(-k^2 / 4 alpha)

  W_ab := - dU_k / d eps_ab = (2 pi / V) sum_k g(k) |rho(k)|^2 / k^2 [ delta_ab - 2 k_a k_b / k^2 (1 + k^2 / 4 alpha) ]

and the random-batch estimate replaces sum_k g(k) by sum_l w_l (w_l = S / P, or the caller's weights):

  W_ab = sum_l (2 pi w_l / V) |rho_l|^2 / k_l^2 [ delta_ab - 2 k_la k_lb / k_l^2 (1 + k_l^2 / 4 alpha) ].

Plain numpy, fp64.  Pin (tests/test_oracle_virial.py): central finite differences of the k-space
energy of an ORTHORHOMBIC box written out from Eq. (2.8) in the test itself, component by component.
"""
from __future__ import annotations

import numpy as np


def kspace_virial(L: float, alpha: float, m, S: float, rho, w=None) -> np.ndarray:
    """float64 [6] = (W_xx, W_yy, W_zz, W_xy, W_xz, W_yz) for the batch m (int [P,3]) and rho ([P,2])."""
    m = np.asarray(m, dtype=np.float64)
    rho = np.asarray(rho, dtype=np.float64)
    P = m.shape[0]
    wl = np.full(P, S / P) if w is None else np.asarray(w, dtype=np.float64)
    V = L ** 3
    k = 2.0 * np.pi * m / L
    k2 = (k ** 2).sum(1)
    pref = 2.0 * np.pi * wl / V * (rho ** 2).sum(1) / k2
    fac = 2.0 / k2 * (1.0 + k2 / (4.0 * alpha))
    out = np.empty(6)
    for n, (a, b) in enumerate(((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2))):
        out[n] = (pref * ((1.0 if a == b else 0.0) - fac * k[:, a] * k[:, b])).sum()
    return out
