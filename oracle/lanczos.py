"""CPU ORACLE for the matrix-free Lanczos spectral bounds -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md P:705: "First, matrix-free Lanczos iterations estimate spectral bounds E_min and E_max";
P:759: ``--lanczos-m 40``.  The paper says no more, so the algorithm is the textbook one (plain
three-term recurrence, no re-orthogonalisation), written out step by step (reading R18):

    v_1 = psi / ||psi||,  beta_0 = 0,  v_0 = 0
    for j = 1..m:   w = H v_j
                    alpha_j = Re <v_j, w>
                    w = w - alpha_j v_j - beta_{j-1} v_{j-1}
                    beta_j = ||w||
                    v_{j+1} = w / beta_j
    T_m = tridiag(beta, alpha, beta);  theta_min, theta_max = extreme eigenvalues of T_m
    c = (theta_max + theta_min)/2,  R = (theta_max - theta_min)/2
    E_min = c - (1 + margin) R,  E_max = c + (1 + margin) R

The Ritz values lie inside the spectrum, so the interval is widened by the relative ``margin``
(BASELINE.json configs[4] quotes its bounds with a factor 1.05: margin = 0.05).  m is capped at D.
Pins (tests/test_oracle_lanczos.py): T_D reproduces the spectrum of a tiny matrix (numpy eigvalsh),
Ritz values are inside the spectrum and converge to its edges, the first Lanczos vectors are
orthonormal, the widened interval encloses the spectrum of the configured GUE.
"""
from __future__ import annotations

import numpy as np


def lanczos_tridiagonal(apply_H, psi, m: int):
    """Return (alpha[0..m-1], beta[0..m-1]) of m Lanczos steps; beta[j] couples v_{j+1} and v_{j+2}."""
    v = np.asarray(psi, dtype=np.complex128).copy()
    m = min(int(m), v.size)
    v /= np.linalg.norm(v)
    v_prev = np.zeros_like(v)
    beta_prev = 0.0
    alpha = np.zeros(m)
    beta = np.zeros(m)
    for j in range(m):
        w = apply_H(v)
        alpha[j] = np.vdot(v, w).real
        w = w - alpha[j] * v - beta_prev * v_prev
        beta[j] = np.linalg.norm(w)
        v_prev, v = v, w / beta[j]
        beta_prev = beta[j]
    return alpha, beta


def ritz_extremes(alpha, beta):
    """Extreme eigenvalues of the m x m tridiagonal T_m (library routine: numpy eigvalsh)."""
    m = len(alpha)
    T = np.diag(np.asarray(alpha, dtype=np.float64))
    for j in range(m - 1):
        T[j, j + 1] = T[j + 1, j] = beta[j]
    ev = np.linalg.eigvalsh(T)
    return float(ev[0]), float(ev[-1])


def lanczos_bounds(apply_H, psi, m: int = 40, margin: float = 0.05):
    """(E_min, E_max, alpha, beta) as defined in the module docstring."""
    alpha, beta = lanczos_tridiagonal(apply_H, psi, m)
    tmin, tmax = ritz_extremes(alpha, beta)
    c, R = 0.5 * (tmax + tmin), 0.5 * (tmax - tmin)
    return c - (1.0 + margin) * R, c + (1.0 + margin) * R, alpha, beta
