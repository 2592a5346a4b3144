"""Pins of the external-block oracle (oracle/external.py; Eq. 10, Eq. 4-5)."""
import numpy as np

import oracle
from paper_2606_31598_b200.inputs import dense_matrix, make_psi


def test_block_loop_equals_the_dense_product():
    D, B = 192, 32
    for herm in (True, False):
        H = dense_matrix(D, 3, hermitian=herm)
        for k in (1, 3):
            Psi = make_psi(D, 5, k=k)
            assert np.allclose(oracle.block_apply(H, B, Psi, "full"), H @ Psi, rtol=0, atol=1e-14)
    H = dense_matrix(D, 3)
    assert np.allclose(H, H.conj().T)
    psi = make_psi(D, 6)
    assert np.allclose(oracle.block_apply(H, B, psi, "pairs"), H @ psi, rtol=0, atol=1e-14)
    assert len(oracle.stored_blocks(6, "pairs")) == 21 and len(oracle.stored_blocks(6, "full")) == 36


def test_pairs_store_needs_a_hermitian_operator():
    D, B = 128, 32
    G = dense_matrix(D, 4, hermitian=False)
    psi = make_psi(D, 7)
    wrong = oracle.block_apply(G, B, psi, "pairs")
    assert np.linalg.norm(wrong - G @ psi) > 0.1 * np.linalg.norm(G @ psi)
    upper = np.triu(G) + np.triu(G, 1).conj().T + 0.0                    # what the pair store represents
    blocks = oracle.block_apply(G, B, psi, "pairs")
    # diagonal blocks are taken whole, so only the strictly-upper BLOCKS are mirrored
    Hm = G.copy()
    for n in range(D // B):
        for m in range(n):
            Hm[n * B:(n + 1) * B, m * B:(m + 1) * B] = G[m * B:(m + 1) * B, n * B:(n + 1) * B].conj().T
    assert np.allclose(blocks, Hm @ psi, rtol=0, atol=1e-14) and upper.shape == G.shape
