"""CPU ORACLE for the Chebyshev propagator e^{-iHt} psi -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Follows PAPER.md Eq. 41-44 step by step:
    c = (E_max + E_min)/2,  R = (E_max - E_min)/2,  H~ = (H - c I)/R
    q_0 = psi,  q_1 = H~ q_0,  q_{l+1} = 2 H~ q_l - q_{l-1}                      (Eq. 41-43)
The paper prints only the recurrence and cites Tal-Ezer & Kosloff (its ref. 3) for the series;
the expansion used is the standard Jacobi-Anger form (reading R7):
    e^{-iHt} psi = e^{-ict} [ J_0(a) q_0 + sum_{l>=1} 2 (-i)^l J_l(a) q_l ],   a = R t.
Truncation (BASELINE.json configs[4]: "terms truncated at |J_k| < 1e-14", R8):
    K = 1 + max{ l : |J_l(a)| >= tol };  terms l = 0..K-1;  K-1 applications of H.

The Bessel table is computed by Miller's backward recurrence normalised with
J_0 + 2 sum_{l>=1} J_{2l} = 1.  Pins: scipy.special.jv, the identity
J_0^2 + 2 sum J_l^2 = 1, the exact eigh propagator at small D, norm conservation and time
reversal (tests/test_oracle_chebyshev.py).  The truncation rule itself is "parity unpinned"
against the paper (the paper's printed order 181 does not pin it).
"""
from __future__ import annotations

import cmath
import math

import numpy as np


def bessel_j_table(a: float, n: int) -> list:
    """[J_0(a), ..., J_{n-1}(a)] for real a by Miller backward recurrence."""
    if a == 0.0:
        return [1.0] + [0.0] * (n - 1)
    x = abs(a)
    start = int(max(n, x) + 30 + 10.0 * math.sqrt(max(n, x)))
    start += start & 1                      # even
    jp1, j = 0.0, 1e-300
    vals = [0.0] * (start + 1)
    vals[start] = j
    for l in range(start, 0, -1):           # J_{l-1} = (2l/x) J_l - J_{l+1}
        jm1 = (2.0 * l / x) * j - jp1
        jp1, j = j, jm1
        vals[l - 1] = j
        if abs(j) > 1e250:                  # rescale to stay finite
            for q in range(l - 1, start + 1):
                vals[q] *= 1e-250
            j *= 1e-250
            jp1 *= 1e-250
    norm = vals[0] + 2.0 * math.fsum(vals[2:start + 1:2])
    out = [v / norm for v in vals[:n]]
    if a < 0:                               # J_l(-x) = (-1)^l J_l(x)
        out = [(-v if (l & 1) else v) for l, v in enumerate(out)]
    return out


def chebyshev_n_terms(a: float, tol: float) -> int:
    """K = 1 + max{l : |J_l(a)| >= tol} (last, not first, crossing: J_l oscillates for l < a)."""
    n = int(abs(a) + 40 + 12.0 * abs(a) ** (1.0 / 3.0) + 40)
    tab = bessel_j_table(a, n)
    assert abs(tab[-1]) < tol and abs(tab[-2]) < tol
    last = 0
    for l, v in enumerate(tab):
        if abs(v) >= tol:
            last = l
    return last + 1


def chebyshev_propagate(apply_H, psi, t: float, e_min: float, e_max: float, tol: float):
    """Return (e^{-iHt} psi, K).  apply_H: callable v -> H v on complex128 numpy vectors."""
    c = 0.5 * (e_max + e_min)
    R = 0.5 * (e_max - e_min)
    a = R * t
    K = chebyshev_n_terms(a, tol)
    J = bessel_j_table(a, K)

    def H_tilde(v):                          # (H - c I)/R applied to v
        return (apply_H(v) - c * v) / R

    q_prev = np.asarray(psi, dtype=np.complex128).copy()       # q_0            Eq. 41
    acc = J[0] * q_prev
    if K > 1:
        q = H_tilde(q_prev)                                    # q_1            Eq. 42
        acc = acc + (2.0 * (-1j) ** 1 * J[1]) * q
        for l in range(1, K - 1):
            q_next = 2.0 * H_tilde(q) - q_prev                 # q_{l+1}        Eq. 43
            acc = acc + (2.0 * (-1j) ** ((l + 1) % 4) * J[l + 1]) * q_next
            q_prev, q = q, q_next
    return cmath.exp(-1j * c * t) * acc, K
