"""CPU ORACLE for an analytically generated Hamiltonian -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md P:159-163 (Eq. 9): "A block may be defined by a formula H^[n,m]_ab = f(n, m, a, b; theta).  The matrix
entries are computed when needed ... the Hamiltonian is defined by the function f and the parameter set theta,
rather than by a stored dense array."  The paper names no f (R22); this build takes a standard dense
model with six parameters theta = (t, alpha, phi, W, beta, delta), a chain with power-law hopping, a Peierls
phase and a quasi-periodic (Aubry-Andre-Harper) potential, written in GLOBAL indices (partition invariant,
P:68-70):

    H_ij = - t exp(+i phi) / (j - i)^alpha     for i < j,
    H_ij = conj(H_ji)                          for i > j,
    H_ii = W cos(2 pi beta i + delta).

The oracle is the definition: the dense matrix from numpy broadcasting in float64 and a plain matmul, row slab
by row slab.  Pins (tests/test_oracle_analytic.py): Hermiticity; alpha = 0, phi = 0, W = 0 is -t (J - I) with the
closed form H psi = -t (sum(psi) - psi); t = 0 is the diagonal potential; large alpha is the nearest-neighbour
tridiagonal chain, whose spectrum W = 0 is -2 t cos(phi + ...) -- checked through the textbook open-chain
eigenvalues -2 t cos(pi m / (D + 1)); the Toeplitz structure H_{i+1,j+1} = H_ij off the diagonal.
"""
from __future__ import annotations

import numpy as np

THETA_KEYS = ("t", "alpha", "phi", "W", "beta", "delta")


def theta_array(theta) -> np.ndarray:
    """theta as the six doubles (t, alpha, phi, W, beta, delta) the C ABI takes."""
    if isinstance(theta, dict):
        return np.array([float(theta[k]) for k in THETA_KEYS], dtype=np.float64)
    th = np.asarray(theta, dtype=np.float64)
    assert th.shape == (6,)
    return th


def analytic_matrix(D: int, theta, i0: int = 0, ni: int | None = None, j0: int = 0, nj: int | None = None) -> np.ndarray:
    """Dense H[i0:i0+ni, j0:j0+nj] as complex128, entry by entry from the formula."""
    t, alpha, phi, W, beta, delta = theta_array(theta)
    ni = D - i0 if ni is None else ni
    nj = D - j0 if nj is None else nj
    i = np.arange(i0, i0 + ni, dtype=np.float64)[:, None]
    j = np.arange(j0, j0 + nj, dtype=np.float64)[None, :]
    d = j - i
    out = np.zeros((ni, nj), dtype=np.complex128)
    up, lo, dg = d > 0, d < 0, d == 0
    mag = np.zeros((ni, nj), dtype=np.float64)
    nz = ~dg
    mag[nz] = t * np.abs(d[nz]) ** (-alpha)
    out[up] = -mag[up] * np.exp(1j * phi)
    out[lo] = -mag[lo] * np.exp(-1j * phi)
    diag = W * np.cos(2.0 * np.pi * beta * (i + 0.0 * j) + delta)
    out[dg] = diag[dg]
    return out


def analytic_apply(D: int, theta, psi, rows=None, slab: int = 1024) -> np.ndarray:
    """phi = H psi ([D] or [D,k]); rows: optional subset of output rows."""
    Psi = np.asarray(psi, dtype=np.complex128)
    one = Psi.ndim == 1
    Psi = Psi.reshape(D, -1)
    if rows is None:
        out = np.empty_like(Psi)
        for i0 in range(0, D, slab):
            n = min(slab, D - i0)
            out[i0:i0 + n] = analytic_matrix(D, theta, i0, n) @ Psi
    else:
        rows = np.asarray(rows, dtype=np.int64)
        out = np.empty((rows.size, Psi.shape[1]), dtype=np.complex128)
        for q, i in enumerate(rows):
            out[q] = analytic_matrix(D, theta, int(i), 1)[0] @ Psi
    return out[:, 0] if one else out
