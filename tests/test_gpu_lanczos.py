"""GPU parity of the NEXT-2 widening: matrix-free Lanczos spectral bounds feeding the
Chebyshev propagator, and multi-step propagation, against the oracle."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import make_psi

pytestmark = pytest.mark.gpu


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(b))


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("mode", ["procedural", "pairs", "full"])
def test_lanczos_coefficients_and_bounds_vs_oracle(mode):
    D, B, m = 2048, 256, 40
    psi = 3.0 * make_psi(D, 99)                       # any non-zero norm: the library normalises
    h = mfh.Hamiltonian(D, B, 21, "c128")
    h.plan(mode)
    e0, e1, alpha, beta = h.lanczos_bounds(to_dev(psi), m=m, margin=0.05)
    H = oracle.materialize(D, 21)
    r0, r1, a_ref, b_ref = oracle.lanczos_bounds(lambda v: H @ v, psi, m=m, margin=0.05)
    # the recurrence amplifies rounding differences step by step: early coefficients agree tightly,
    # the extreme Ritz values (what the method uses) are insensitive
    assert np.allclose(alpha[:12], a_ref[:12], rtol=0, atol=1e-10)
    assert np.allclose(beta[:12], b_ref[:12], rtol=1e-10, atol=0)
    assert abs(e0 - r0) < 1e-8 and abs(e1 - r1) < 1e-8
    ev = np.linalg.eigvalsh(H)
    assert e0 < ev[0] and e1 > ev[-1]                 # the widened interval encloses the spectrum


def test_lanczos_bounds_feed_the_chebyshev_propagator():
    D, B, t = 1024, 256, 20.0
    psi = make_psi(D, 99)
    h = mfh.Hamiltonian(D, B, 21, "c128")
    h.plan("procedural")
    d_psi = to_dev(psi)
    e0, e1, _, _ = h.lanczos_bounds(d_psi, m=40, margin=0.05)
    out, K = h.chebyshev(d_psi, t, e0, e1, 1e-14)
    H = oracle.materialize(D, 21)
    w, U = np.linalg.eigh(H)
    exact = U @ (np.exp(-1j * w * t) * (U.conj().T @ psi))
    assert rel_l2(out.cpu().numpy(), exact) <= 1e-11
    ref, K_ref = oracle.chebyshev_propagate(lambda v: H @ v, psi, t, e0, e1, 1e-14)
    assert K == K_ref and rel_l2(out.cpu().numpy(), ref) <= 1e-11


def test_multi_step_propagation_is_the_group_product():
    D, B, tau, n = 1024, 256, 1.7, 5
    psi = make_psi(D, 4)
    h = mfh.Hamiltonian(D, B, 21, "c128")
    h.plan("procedural")
    out, K = h.chebyshev_steps(to_dev(psi), tau, n, -2.1, 2.1, 1e-14)
    H = oracle.materialize(D, 21)
    ref = psi
    for _ in range(n):                                 # the oracle, step by step
        ref, K_ref = oracle.chebyshev_propagate(lambda v: H @ v, ref, tau, -2.1, 2.1, 1e-14)
    assert K == K_ref and rel_l2(out.cpu().numpy(), ref) <= 1e-11
    w, U = np.linalg.eigh(H)                           # U(tau)^n = U(n tau)
    exact = U @ (np.exp(-1j * w * tau * n) * (U.conj().T @ psi))
    assert rel_l2(out.cpu().numpy(), exact) <= 1e-11
    assert abs(np.linalg.norm(out.cpu().numpy()) - 1.0) <= 1e-12


def test_lanczos_argument_errors_and_c64():
    D, B = 1024, 256
    psi = make_psi(D, 1, dtype="c64")
    h = mfh.Hamiltonian(D, B, 21, "c64")
    with pytest.raises(mfh.MfhError) as e:
        h.lanczos_bounds(to_dev(psi))
    assert e.value.code == mfh.MFH_ERR_BAD_STATE
    h.plan("procedural")
    with pytest.raises(mfh.MfhError) as e:
        h.lanczos_bounds(to_dev(psi), m=0)
    assert e.value.code == mfh.MFH_ERR_INVALID_ARG
    e0, e1, alpha, beta = h.lanczos_bounds(to_dev(psi), m=30, margin=0.05)
    H = oracle.materialize(D, 21)
    r0, r1, _, _ = oracle.lanczos_bounds(lambda v: H @ v, psi.astype(np.complex128), m=30, margin=0.05)
    assert abs(e0 - r0) < 1e-4 and abs(e1 - r1) < 1e-4
