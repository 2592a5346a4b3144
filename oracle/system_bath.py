"""CPU ORACLE for the system-bath Hamiltonian action -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md P:676-690:  H = H_S (x) I_B + I_S (x) H_B + g sum_a A_a (x) B_a  acting on w in C^{d_S} (x) C^{d_B}
"without constructing the full D x D Hamiltonian"; the paper's run has one interaction operator, so each
application uses two dense bath-side operators H_B and B_1 applied to R = d_S simultaneous state
components (Eq. 12).  With the state stored as X[b][s] (bath index b, system index s: the
k-vector layout [D][k] of the library with D = d_B, k = d_S) the definition reads, entry by entry,

    Y[b][s] = sum_s' H_S[s][s'] X[b][s']  +  sum_b' H_B[b][b'] X[b'][s]
              + g sum_s' A[s][s'] sum_b' B_1[b][b'] X[b'][s'].

The paper does not give H_S, A or the distribution of the bath operators (R19): H_B and B_1
are the seeded GUE of BASELINE.json (d_B x d_B, entry rule of mfh_oracle.c, two seeds), H_S and A are
small Hermitian matrices passed in.  Pins (tests/test_oracle_system_bath.py): the explicit Kronecker
matrix at tiny sizes (numpy kron + matmul), Hermiticity, the g = 0 and H_S = 0 special cases.
"""
from __future__ import annotations

import numpy as np

from . import apply as _apply


def sb_apply(d_B: int, B: int, seed_HB: int, seed_B1: int, H_S, A, g: float, X, rows=None) -> np.ndarray:
    """Y = (H w) in the [d_B][d_S] layout; rows: optional subset of bath indices b."""
    X = np.ascontiguousarray(X, dtype=np.complex128)
    d_S = X.shape[1]
    H_S = np.asarray(H_S, dtype=np.complex128).reshape(d_S, d_S)
    A = np.asarray(A, dtype=np.complex128).reshape(d_S, d_S)
    Y1 = _apply(d_B, B, seed_HB, X, rows=rows)            # (H_B X)[b][s]
    Y2 = _apply(d_B, B, seed_B1, X, rows=rows)            # (B_1 X)[b][s']
    Xr = X if rows is None else X[np.asarray(rows)]
    out = np.empty_like(Y1)
    for s in range(d_S):                                   # the definition, term by term
        acc = Y1[:, s].copy()
        for sp in range(d_S):
            acc += H_S[s, sp] * Xr[:, sp] + g * A[s, sp] * Y2[:, sp]
        out[:, s] = acc
    return out
