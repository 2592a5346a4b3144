"""Pins for the oracle's Chebyshev propagator (Eq. 41-44).

Bessel table vs scipy and two classical identities; the propagator vs the exact
U exp(-i Lambda t) U^dagger psi from eigh; unitarity (Eq. 40); time reversal; the term
count of BASELINE.json configs[4]; and the divergence of the literal +-sqrt(2)*1.05 bounds
(SURVEY.md finding 1, reading R8).
"""
import numpy as np
import pytest
import scipy.special

import oracle
from paper_2606_31598_b200.inputs import make_psi


@pytest.mark.parametrize("a", [0.0, 0.3, 7.5, 74.25, 105.0, -12.0])
def test_bessel_table(a):
    n = 220
    J = np.array(oracle.bessel_j_table(a, n))
    ref = scipy.special.jv(np.arange(n), a)
    assert np.max(np.abs(J - ref)) < 5e-15   # scipy itself is good to a few 1e-16 relative
    assert abs(J[0] + 2 * J[2::2].sum() - 1.0) < 1e-14           # generating-function identity
    assert abs(J[0] ** 2 + 2 * (J[1:] ** 2).sum() - 1.0) < 1e-14  # Parseval identity


def test_term_count_of_config5():
    """a = R t = 2.1 * 50 = 105, tol 1e-14 -> K = 152; last-crossing rule."""
    assert oracle.chebyshev_n_terms(105.0, 1e-14) == 152
    assert oracle.chebyshev_n_terms(100.0, 1e-14) == 147
    assert oracle.chebyshev_n_terms(74.25, 1e-14) == 117
    assert oracle.chebyshev_n_terms(0.0, 1e-14) == 1
    J = scipy.special.jv(np.arange(400), 105.0)
    assert abs(J[151]) >= 1e-14 and np.all(np.abs(J[152:]) < 1e-14)
    assert np.count_nonzero(np.diff(np.sign(J[:100]))) > 20   # J_k oscillates through 0 below k=a


@pytest.mark.parametrize("D,t", [(128, 3.0), (512, 50.0)])
def test_propagator_against_eigh(D, t):
    seed, B = 21, 64
    H = oracle.materialize(D, seed)
    psi = make_psi(D, 99)
    w, U = np.linalg.eigh(H)
    exact = U @ (np.exp(-1j * w * t) * (U.conj().T @ psi))
    out, K = oracle.chebyshev_propagate(lambda v: oracle.apply(D, B, seed, v), psi, t, -2.1, 2.1, 1e-14)
    assert K == oracle.chebyshev_n_terms(2.1 * t, 1e-14)
    assert np.linalg.norm(out - exact) < 2e-13
    assert abs(np.linalg.norm(out) - 1.0) < 1e-12


def test_off_centre_bounds_and_time_reversal():
    """c != 0 exercises the e^{-ict} phase and the (H - c)/R shift; e^{+iHt} e^{-iHt} psi = psi."""
    D, seed, B, t = 256, 5, 64, 7.0
    H = oracle.materialize(D, seed)
    psi = make_psi(D, 4)
    f = lambda v: H @ v
    w, U = np.linalg.eigh(H)
    exact = U @ (np.exp(-1j * w * t) * (U.conj().T @ psi))
    out, _ = oracle.chebyshev_propagate(f, psi, t, -2.3, 2.6, 1e-14)
    assert np.linalg.norm(out - exact) < 1e-13
    back, _ = oracle.chebyshev_propagate(f, out, -t, -2.3, 2.6, 1e-14)
    assert np.linalg.norm(back - psi) < 2e-13


def test_literal_config5_bounds_diverge():
    """+-sqrt(2)*1.05 lies inside the spectrum [-2,2] of this GUE, so T_k grows exponentially."""
    D, seed, t = 256, 21, 50.0
    H = oracle.materialize(D, seed)
    psi = make_psi(D, 99)
    b = np.sqrt(2.0) * 1.05
    out, _ = oracle.chebyshev_propagate(lambda v: H @ v, psi, t, -b, b, 1e-14)
    assert abs(np.linalg.norm(out) - 1.0) > 1e6
