"""CPU ORACLE for externally stored blocks -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md P:165-169 (Eq. 10): "A block may be stored outside GPU memory and retrieved by key:
H^[n,m] = D[key(n,m)] ... The computational kernel remains unchanged."  The operator is whatever dense array the
caller holds; the oracle is the two-level product of Eq. 4-5 / Eq. 7 written out over the blocks of that array,

    phi^[n] = sum_m H^[n,m] psi^[m],        H^[n,m] = H[n B:(n+1) B, m B:(m+1) B],

one numpy matmul per block in complex128.  `store` names which blocks a plan keeps: "full" = all N_blk^2 of them,
"pairs" = the canonical blocks n <= m of a Hermitian operator, the other positions served by the conjugate
transpose.  Pin (tests/test_oracle_external.py): the plain dense product H @ psi, for Hermitian and
general matrices, and the failure of "pairs" on a non-Hermitian matrix.
"""
from __future__ import annotations

import numpy as np


def stored_blocks(n_blk: int, store: str):
    """Keys (n, m) of the blocks a plan stores."""
    assert store in ("full", "pairs")
    return [(n, m) for n in range(n_blk) for m in range(n_blk) if store == "full" or n <= m]


def block_apply(H, B: int, psi, store: str = "full") -> np.ndarray:
    """phi = H psi from the stored blocks of the dense array H ([D, D]); psi: [D] or [D, k]."""
    H = np.asarray(H, dtype=np.complex128)
    D = H.shape[0]
    assert H.shape == (D, D) and D % B == 0
    n_blk = D // B
    Psi = np.asarray(psi, dtype=np.complex128)
    one = Psi.ndim == 1
    Psi = Psi.reshape(D, -1)
    out = np.zeros_like(Psi)
    for (n, m) in stored_blocks(n_blk, store):
        blk = H[n * B:(n + 1) * B, m * B:(m + 1) * B]
        out[n * B:(n + 1) * B] += blk @ Psi[m * B:(m + 1) * B]
        if store == "pairs" and n != m:                       # the mirrored position from the same stored block
            out[m * B:(m + 1) * B] += blk.conj().T @ Psi[n * B:(n + 1) * B]
    return out[:, 0] if one else out
