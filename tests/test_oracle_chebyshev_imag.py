"""Pins of the oracle's imaginary-time Chebyshev filter e^{-beta (H - E_min)} psi (oracle/chebyshev.py;
PAPER.md P:784-790 names the filter, Eq. 41-43 give the recurrence; R21)."""
import numpy as np
import pytest
import scipy.special

import oracle
from paper_2606_31598_b200.inputs import make_psi


@pytest.mark.parametrize("a", [0.0, 0.4, 7.5, 71.3, 300.0, -9.0])
def test_scaled_bessel_i_table(a):
    n = 200
    tab = np.array(oracle.bessel_i_scaled_table(a, n))
    ref = scipy.special.ive(np.arange(n), a)                  # e^{-|a|} I_l(a)
    assert np.max(np.abs(tab - ref)) < 1e-15 + 4e-15 * np.max(np.abs(ref))
    full = np.array(oracle.bessel_i_scaled_table(abs(a), 900))
    assert abs(full[0] + 2.0 * full[1:].sum() - 1.0) < 1e-13  # e^{-x} (I_0 + 2 sum I_l) = 1


def test_series_reproduces_the_scalar_exponential():
    """The expansion itself, on numbers: e^{-a x} = I_0(a) + 2 sum (-1)^l I_l(a) T_l(x), |x| <= 1."""
    a = 12.5
    K = oracle.chebyshev_imag_n_terms(a, 1e-15)
    Isc = np.array(oracle.bessel_i_scaled_table(a, K))
    x = np.linspace(-1, 1, 41)
    T = np.cos(np.outer(np.arange(K), np.arccos(x)))
    coef = np.where(np.arange(K) == 0, 1.0, 2.0) * (-1.0) ** np.arange(K) * Isc
    assert np.max(np.abs(coef @ T - np.exp(-a * x - a))) < 1e-14


@pytest.mark.parametrize("D,beta", [(128, 0.2), (256, 3.0), (512, 20.0)])
def test_filter_against_eigh(D, beta):
    seed, B = 21, 64
    H = oracle.materialize(D, seed)
    psi = make_psi(D, 5)
    w, U = np.linalg.eigh(H)
    e_min, e_max = -2.3, 2.2                                   # off-centre bounds enclosing the spectrum
    assert e_min < w[0] and w[-1] < e_max
    ref = U @ (np.exp(-beta * (w - e_min)) * (U.conj().T @ psi))
    out, K = oracle.chebyshev_imag_propagate(lambda v: oracle.apply(D, B, seed, v), psi, beta, e_min, e_max, 1e-14)
    assert np.linalg.norm(out - ref) <= 1e-12 * np.linalg.norm(psi)
    assert K == oracle.chebyshev_imag_n_terms(0.5 * (e_max - e_min) * beta, 1e-14)


def test_semigroup_identity_and_beta_zero():
    D, seed, B = 128, 21, 32
    psi = make_psi(D, 6)
    ap = lambda v: oracle.apply(D, B, seed, v)                 # noqa: E731
    o0, K0 = oracle.chebyshev_imag_propagate(ap, psi, 0.0, -2.1, 2.1, 1e-14)
    assert K0 == 1 and np.array_equal(o0, psi)
    a, _ = oracle.chebyshev_imag_propagate(ap, psi, 1.5, -2.1, 2.1, 1e-15)
    b, _ = oracle.chebyshev_imag_propagate(ap, a, 2.5, -2.1, 2.1, 1e-15)
    c, _ = oracle.chebyshev_imag_propagate(ap, psi, 4.0, -2.1, 2.1, 1e-15)
    assert np.linalg.norm(b - c) <= 1e-13
    assert np.linalg.norm(c) < np.linalg.norm(a) < 1.0         # e^{-beta (H - E_min)} is a contraction


def test_order_grows_like_sqrt_of_the_argument():
    """K - 1 ~ sqrt(2 a ln(2/tol)) for large a (Gaussian tail of e^{-a} I_l(a)); at the paper's filter
    argument a = R beta / 2 = 713 * 0.2 / 2 = 71.3 the rule gives an order below the 80 the paper
    used as an input parameter."""
    K = oracle.chebyshev_imag_n_terms(71.3, 1e-7)
    assert 40 <= K - 1 <= 80
    assert abs((K - 1) - np.sqrt(2 * 71.3 * np.log(2 / 1e-7))) < 6
