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


# ---- imaginary time (SURVEY 8f "later": the paper's TPQ filter e^{-beta H/2}) ------------------
# The paper names the filter ("the imaginary-time TPQ Chebyshev filter used order 80") without printing its
# series.  With the SAME recurrence (Eq. 41-43) the standard expansion is the modified-Bessel analogue of
# Jacobi-Anger, e^{-a x} = I_0(a) + 2 sum_{l>=1} (-1)^l I_l(a) T_l(x) for |x| <= 1, so with a = R beta
#     e^{-beta H} psi = e^{-beta c} [ I_0(a) q_0 + sum_{l>=1} 2 (-1)^l I_l(a) q_l ].
# I_l(a) grows like e^a; the oracle (and the library) work with the scaled values e^{-a} I_l(a) and return
#     out = e^{-beta (H - E_min)} psi = sum_l (2 - delta_l0) (-1)^l [e^{-a} I_l(a)] q_l      (c - R = E_min)
# whose largest eigen-factor is <= 1; e^{-beta H} psi = e^{-beta E_min} out.
# Truncation (R21, parity unpinned against the paper, whose order is an input parameter):
#     K = 1 + max{ l : 2 e^{-a} I_l(a) >= tol }.

def bessel_i_scaled_table(a: float, n: int) -> list:
    """[e^{-|a|} I_0(a), ..., e^{-|a|} I_{n-1}(a)] by Miller backward recurrence
    I_{l-1} = (2l/x) I_l + I_{l+1}, normalised with e^{-x} (I_0 + 2 sum_{l>=1} I_l) = 1."""
    if a == 0.0:
        return [1.0] + [0.0] * (n - 1)
    x = abs(a)
    start = int(max(n, x) + 30 + 10.0 * math.sqrt(max(n, x)))
    ip1, i = 0.0, 1e-300
    vals = [0.0] * (start + 1)
    vals[start] = i
    for l in range(start, 0, -1):
        im1 = (2.0 * l / x) * i + ip1
        ip1, i = i, im1
        vals[l - 1] = i
        if abs(i) > 1e250:
            for q in range(l - 1, start + 1):
                vals[q] *= 1e-250
            i *= 1e-250
            ip1 *= 1e-250
    norm = vals[0] + 2.0 * math.fsum(vals[1:])
    out = [v / norm for v in vals[:n]]
    if a < 0:                               # I_l(-x) = (-1)^l I_l(x)
        out = [(-v if (l & 1) else v) for l, v in enumerate(out)]
    return out


def chebyshev_imag_n_terms(a: float, tol: float) -> int:
    n = int(abs(a) + 60 + 12.0 * math.sqrt(abs(a) * 40.0 + 1.0))
    tab = bessel_i_scaled_table(abs(a), n)
    assert 2.0 * tab[-1] < tol
    last = 0
    for l, v in enumerate(tab):
        if 2.0 * v >= tol:
            last = l
    return last + 1


def chebyshev_imag_propagate(apply_H, psi, beta: float, e_min: float, e_max: float, tol: float):
    """Return (e^{-beta (H - e_min)} psi, K), beta >= 0.  apply_H: callable v -> H v."""
    c = 0.5 * (e_max + e_min)
    R = 0.5 * (e_max - e_min)
    a = R * beta
    K = chebyshev_imag_n_terms(a, tol)
    Isc = bessel_i_scaled_table(a, K)

    def H_tilde(v):
        return (apply_H(v) - c * v) / R

    q_prev = np.asarray(psi, dtype=np.complex128).copy()       # q_0            Eq. 41
    acc = Isc[0] * q_prev
    if K > 1:
        q = H_tilde(q_prev)                                    # q_1            Eq. 42
        acc = acc - 2.0 * Isc[1] * q
        for l in range(1, K - 1):
            q_next = 2.0 * H_tilde(q) - q_prev                 # q_{l+1}        Eq. 43
            acc = acc + (2.0 * (-1.0) ** (l + 1) * Isc[l + 1]) * q_next
            q_prev, q = q, q_next
    return acc, K
