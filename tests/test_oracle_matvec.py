"""Pins for the oracle's H psi: explicit dense matmul, partition invariance, Hermiticity of the
operator, GUE spectrum (semicircle edge at +-2), linearity and the coupling-scan special cases.

PAPER.md Eq. 4-5 says the block product IS the dense product; Eq. 7 is
the loop; P:68-70 / P:828-836 demand partition invariance; P:178-181 the Hermitian relation.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2606_31598_b200.inputs import lambda_grid, make_psi


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.mark.parametrize("D,B", [(64, 16), (256, 64), (1024, 128)])
def test_apply_equals_dense_matmul(D, B):
    """Materialise D x D with the entry rule, multiply with numpy (library special case) and
    with an explicit triple loop at the smallest size (brute force)."""
    seed = 1234
    H = oracle.materialize(D, seed)
    psi = make_psi(D, 99)
    phi = oracle.apply(D, B, seed, psi)
    assert _rel(phi, H @ psi) < 1e-14
    if D == 64:
        brute = np.zeros(D, dtype=np.complex128)
        for i in range(D):
            for j in range(D):
                brute[i] += oracle.entry(D, seed, i, j) * psi[j]
        assert _rel(phi, brute) < 1e-14


def test_config1_against_dense_matmul():
    """BASELINE.json configs[0]: D=4096, B=512, seed 1234, psi seed 99, vs explicit dense matmul."""
    D, B, seed = 4096, 512, 1234
    psi = make_psi(D, 99)
    rows = np.arange(0, D, 37)
    phi_rows = oracle.apply(D, B, seed, psi, rows=rows)
    H_rows = np.concatenate([oracle.materialize(D, seed, int(i), 1) for i in rows], axis=0)
    assert _rel(phi_rows, H_rows @ psi) < 1e-14
    # ||H psi||^2 -> tr H^2 / D = 1 for a random normalised psi
    assert abs(np.linalg.norm(phi_rows) ** 2 * D / rows.size - 1.0) < 0.3


def test_partition_invariance():
    """Changing N_blk must not change the operator."""
    D, seed = 512, 5
    psi = make_psi(D, 1)
    ref = oracle.apply(D, D, seed, psi)
    for B in (1, 8, 64, 256):
        assert _rel(oracle.apply(D, B, seed, psi), ref) < 1e-15


def test_row_subset_matches_full():
    D, B, seed = 512, 64, 9
    psi = make_psi(D, 2)
    full = oracle.apply(D, B, seed, psi)
    rows = np.array([0, 3, 63, 64, 200, 511])
    assert np.array_equal(oracle.apply(D, B, seed, psi, rows=rows), full[rows])


def test_operator_hermiticity():
    """<a|H b> = conj(<b|H a>) to 1e-13 (BASELINE.json north_star)."""
    D, B, seed = 1024, 128, 21
    a, b = make_psi(D, 10), make_psi(D, 11)
    lhs = np.vdot(a, oracle.apply(D, B, seed, b))
    rhs = np.conj(np.vdot(b, oracle.apply(D, B, seed, a)))
    assert abs(lhs - rhs) < 1e-13
    assert abs(np.vdot(a, oracle.apply(D, B, seed, a)).imag) < 1e-13


def test_linearity():
    D, B, seed = 256, 32, 4
    a, b = make_psi(D, 1), make_psi(D, 2)
    z = 0.3 - 1.7j
    lhs = oracle.apply(D, B, seed, a + z * b)
    rhs = oracle.apply(D, B, seed, a) + z * oracle.apply(D, B, seed, b)
    assert _rel(lhs, rhs) < 1e-14


@pytest.mark.parametrize("D", [256, 1024])
def test_gue_spectrum_semicircle(D):
    """E|H_ij|^2 = 1/D  =>  semicircle on [-2,2]: tr H^2/D -> 1, tr H^4/D -> 2 (Catalan),
    extreme eigenvalues at +-2 within a few D^{-2/3} (Tracy-Widom scale)."""
    H = oracle.materialize(D, 1234)
    w = np.linalg.eigvalsh(H)
    assert abs((w ** 2).mean() - 1.0) < 4.0 / D + 0.01
    assert abs((w ** 4).mean() - 2.0) < 0.05
    tw = 4.0 * D ** (-2.0 / 3.0)
    assert abs(w[-1] - 2.0) < tw and abs(w[0] + 2.0) < tw
    # semicircle CDF at 0 and at 1: 1/2 and 1/2 + (sqrt(3)/2 + 2 pi/3... ) closed form below
    F1 = 0.5 + (1.0 * math.sqrt(4 - 1.0) / 4 + math.asin(0.5)) / math.pi
    assert abs((w < 0).mean() - 0.5) < 0.02 and abs((w < 1.0).mean() - F1) < 0.02


def test_multi_vector_equals_single_vectors():
    D, B, seed, k = 256, 64, 8, 5
    Psi = make_psi(D, 9, k=k)
    Phi = oracle.apply(D, B, seed, Psi)
    for v in range(k):
        assert _rel(Phi[:, v], oracle.apply(D, B, seed, Psi[:, v].copy())) < 1e-15


def test_coupling_scan_special_cases():
    """Phi_v = h0 (.) psi_v + lambda_v V psi_v; lambda=0 column is h0 (.) psi (textbook case);
    every column equals the dense (diag(h0) + lambda V) psi."""
    D, B, k = 256, 64, 4
    lam = lambda_grid(k)
    assert lam[0] == 0.0 and lam[-1] == 2.0 and np.allclose(np.diff(lam), 2.0 / (k - 1))
    Psi = make_psi(D, 9, k=k)
    Phi = oracle.apply_scan(D, B, 8, 7, lam, Psi)
    h0 = oracle.h0_diagonal(D, 7)
    V = oracle.materialize(D, 8)
    assert _rel(Phi[:, 0], h0 * Psi[:, 0]) < 1e-15
    for v in range(k):
        dense = (np.diag(h0) + lam[v] * V) @ Psi[:, v]
        assert _rel(Phi[:, v], dense) < 1e-14
    rows = np.array([1, 100, 255])
    assert np.array_equal(oracle.apply_scan(D, B, 8, 7, lam, Psi, rows=rows), Phi[rows])


def test_c64_inputs_are_evaluated_in_double():
    """c64 oracle = the same mathematical H in double on the float-rounded psi (R6)."""
    D, B, seed = 256, 64, 8
    psi32 = make_psi(D, 9, dtype="c64")
    assert psi32.dtype == np.complex64
    phi = oracle.apply(D, B, seed, psi32)
    assert phi.dtype == np.complex128
    assert _rel(phi, oracle.materialize(D, seed) @ psi32.astype(np.complex128)) < 1e-14
