"""Pins of the Lanczos-bounds oracle (oracle/lanczos.py; R18)."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200.inputs import make_psi


def test_full_lanczos_reproduces_the_spectrum_of_a_tiny_matrix():
    # m = D steps: T_D is unitarily similar to H (exact arithmetic); at D = 24 rounding leaves 1e-9
    D = 24
    H = oracle.materialize(D, 5)
    alpha, beta = oracle.lanczos_tridiagonal(lambda v: H @ v, make_psi(D, 3), D)
    T = np.diag(alpha) + np.diag(beta[:-1], 1) + np.diag(beta[:-1], -1)
    assert np.allclose(np.linalg.eigvalsh(T), np.linalg.eigvalsh(H), atol=1e-8)


def test_first_lanczos_vectors_are_orthonormal_and_tridiagonalise():
    D, m = 256, 12
    H = oracle.materialize(D, 21)
    psi = make_psi(D, 99)
    alpha, beta = oracle.lanczos_tridiagonal(lambda v: H @ v, psi, m)
    V = [psi / np.linalg.norm(psi)]                      # rebuild the basis from the coefficients alone
    prev, b_prev = np.zeros(D, complex), 0.0
    for j in range(m - 1):
        w = H @ V[j] - alpha[j] * V[j] - b_prev * prev
        prev, b_prev = V[j], beta[j]
        V.append(w / beta[j])
    V = np.stack(V, axis=1)
    assert np.allclose(V.conj().T @ V, np.eye(m), atol=1e-10)
    T = V.conj().T @ H @ V
    assert np.allclose(np.diag(T).real, alpha, atol=1e-12)
    assert np.allclose(np.abs(np.diag(T, 1)), beta[:m - 1], atol=1e-10)
    assert np.abs(np.triu(T, 2)).max() < 1e-10


@pytest.mark.parametrize("D", [512, 2048])
def test_ritz_values_inside_the_spectrum_and_widened_bounds_enclose_it(D):
    H = oracle.materialize(D, 21)
    ev = np.linalg.eigvalsh(H)
    e_min, e_max, alpha, beta = oracle.lanczos_bounds(lambda v: H @ v, make_psi(D, 99), m=40, margin=0.05)
    tmin, tmax = oracle.ritz_extremes(alpha, beta)
    assert ev[0] - 1e-12 <= tmin and tmax <= ev[-1] + 1e-12          # Ritz values never leave the spectrum
    assert tmin - ev[0] < 0.03 * 4.0 and ev[-1] - tmax < 0.03 * 4.0   # and are within 3 % of the width of its edges
    assert e_min < ev[0] and e_max > ev[-1]                           # 5 % margin encloses the spectrum
    assert abs(e_max - 2.1) < 0.08 and abs(e_min + 2.1) < 0.08        # GUE edge 2 (c-4): bounds ~ +-2.1


def test_m_is_capped_at_the_dimension_and_shifted_scaled_operators():
    D = 32
    H = oracle.materialize(D, 7)
    alpha, beta = oracle.lanczos_tridiagonal(lambda v: H @ v, make_psi(D, 1), 40)
    assert len(alpha) == D
    # Lanczos is equivariant under H -> a H + b: alpha -> a alpha + b, beta -> |a| beta
    a2, b2 = oracle.lanczos_tridiagonal(lambda v: 3.0 * (H @ v) + 0.5 * v, make_psi(D, 1), 10)
    assert np.allclose(a2, 3.0 * alpha[:10] + 0.5, atol=1e-10) and np.allclose(b2, 3.0 * beta[:10], atol=1e-10)
