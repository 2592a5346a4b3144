"""Pins of the analytic-source oracle (oracle/analytic.py; Eq. 9; R22)."""
import numpy as np

import oracle
from paper_2606_31598_b200.inputs import make_psi

TH = dict(t=0.7, alpha=1.3, phi=0.4, W=1.1, beta=(np.sqrt(5.0) - 1.0) / 2.0, delta=0.25)


def test_hermitian_toeplitz_off_diagonal_and_block_views():
    D = 96
    H = oracle.analytic_matrix(D, TH)
    assert np.array_equal(H, H.conj().T) and np.all(H.imag.diagonal() == 0.0)
    off = H - np.diag(H.diagonal())
    assert np.array_equal(off[1:, 1:], off[:-1, :-1])                       # depends on j - i only
    assert np.array_equal(oracle.analytic_matrix(D, TH, 32, 16, 64, 32), H[32:48, 64:96])
    assert np.isclose(H[3, 10], -0.7 * np.exp(0.4j) / 7.0 ** 1.3) and np.isclose(H[10, 3], np.conj(H[3, 10]))
    assert np.isclose(H[5, 5], 1.1 * np.cos(2 * np.pi * TH["beta"] * 5 + 0.25))


def test_all_to_all_closed_form():
    """alpha = 0, phi = 0, W = 0: H = -t (J - I), so H psi = -t (sum(psi) - psi)."""
    D = 200
    psi = make_psi(D, 1)
    th = dict(TH, alpha=0.0, phi=0.0, W=0.0)
    assert np.allclose(oracle.analytic_apply(D, th, psi), -0.7 * (psi.sum() - psi), rtol=0, atol=1e-13)


def test_diagonal_only_and_linearity():
    D = 128
    psi, chi = make_psi(D, 2), make_psi(D, 3)
    th = dict(TH, t=0.0)
    pot = 1.1 * np.cos(2 * np.pi * TH["beta"] * np.arange(D) + 0.25)
    assert np.allclose(oracle.analytic_apply(D, th, psi), pot * psi, rtol=0, atol=1e-15)
    a = oracle.analytic_apply(D, TH, psi + 2j * chi)
    b = oracle.analytic_apply(D, TH, psi) + 2j * oracle.analytic_apply(D, TH, chi)
    assert np.allclose(a, b, rtol=0, atol=1e-13)


def test_nearest_neighbour_limit_has_the_open_chain_spectrum():
    """alpha -> infinity leaves the tridiagonal chain; with W = 0 its eigenvalues are -2 t cos(pi m / (D + 1))
    whatever the Peierls phase (a gauge transformation on an open chain)."""
    D = 64
    th = dict(TH, alpha=60.0, W=0.0)
    ev = np.linalg.eigvalsh(oracle.analytic_matrix(D, th))
    ref = np.sort(-2 * 0.7 * np.cos(np.pi * np.arange(1, D + 1) / (D + 1)))
    assert np.allclose(ev, ref, rtol=0, atol=1e-12)


def test_row_subset_k_vectors_and_dense_matmul():
    D = 300
    Psi = make_psi(D, 4, k=3)
    H = oracle.analytic_matrix(D, TH)
    full = oracle.analytic_apply(D, TH, Psi, slab=128)
    assert np.allclose(full, H @ Psi, rtol=0, atol=1e-13)
    rows = np.array([0, 7, 150, 299])
    assert np.allclose(oracle.analytic_apply(D, TH, Psi, rows=rows), full[rows], rtol=0, atol=1e-13)
    a, b = make_psi(D, 5), make_psi(D, 6)
    assert abs(np.vdot(a, H @ b) - np.conj(np.vdot(b, H @ a))) < 1e-13
