"""Pins of the system-bath oracle (oracle/system_bath.py; R19)."""
import numpy as np

import oracle
from paper_2606_31598_b200.inputs import make_psi, small_hermitian


def _setup(d_B=64, d_S=4, B=16):
    H_S, A = small_hermitian(d_S, 33), small_hermitian(d_S, 34)
    X = make_psi(d_B, 35, k=d_S)
    return d_B, d_S, B, H_S, A, X


def test_equals_the_explicit_kronecker_matrix():
    d_B, d_S, B, H_S, A, X = _setup()
    g = 0.37
    HB, B1 = oracle.materialize(d_B, 31), oracle.materialize(d_B, 32)
    # w index = s * d_B + b  (C^{d_S} (x) C^{d_B}); X[b][s] = w[s * d_B + b]
    H = np.kron(H_S, np.eye(d_B)) + np.kron(np.eye(d_S), HB) + g * np.kron(A, B1)
    w = X.T.reshape(-1)
    ref = (H @ w).reshape(d_S, d_B).T
    Y = oracle.sb_apply(d_B, B, 31, 32, H_S, A, g, X)
    assert np.allclose(Y, ref, rtol=0, atol=1e-13)
    assert np.allclose(H, H.conj().T)                       # the composite operator is Hermitian


def test_special_cases_and_row_subset():
    d_B, d_S, B, H_S, A, X = _setup()
    Z = np.zeros((d_S, d_S))
    Y0 = oracle.sb_apply(d_B, B, 31, 32, Z, A, 0.0, X)      # g = 0, H_S = 0: just H_B on every column
    assert np.allclose(Y0, oracle.apply(d_B, B, 31, X), atol=1e-14)
    Y1 = oracle.sb_apply(d_B, B, 31, 32, H_S, A, 0.0, X)    # g = 0: bath and system decouple
    assert np.allclose(Y1 - Y0, X @ H_S.T, atol=1e-14)
    rows = np.array([0, 5, 17, 63])
    Yr = oracle.sb_apply(d_B, B, 31, 32, H_S, A, 0.8, X, rows=rows)
    assert np.allclose(Yr, oracle.sb_apply(d_B, B, 31, 32, H_S, A, 0.8, X)[rows], atol=1e-14)


def test_hermiticity_of_the_action():
    d_B, d_S, B, H_S, A, X = _setup()
    Z = make_psi(d_B, 36, k=d_S)
    HX = oracle.sb_apply(d_B, B, 31, 32, H_S, A, 0.6, X)
    HZ = oracle.sb_apply(d_B, B, 31, 32, H_S, A, 0.6, Z)
    assert abs(np.vdot(Z, HX) - np.conj(np.vdot(X, HZ))) < 1e-13
