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


@pytest.mark.parametrize("dtype,mode", [("c128", "procedural"), ("c128", "full"), ("c64", "procedural"), ("c64", "full"), ("c64", "pairs")])
def test_coupling_scan_propagation_k_columns(dtype, mode):
    """mfh_chebyshev_scan: k states propagated under k Hamiltonians H_v = diag(h0) + lambda_v V at once (one k-vector
    plan, every block generated or read once per term), against the exact eigh propagator of each H_v and the
    oracle's step-by-step series."""
    from paper_2606_31598_b200.inputs import lambda_grid
    D, B, k, t = 1024, 128, 4, 2.5
    lam = lambda_grid(k)                                   # 0, 2/3, 4/3, 2
    Psi = make_psi(D, 9, k=k, dtype=dtype)
    h = mfh.Hamiltonian(D, B, 8, dtype, kind="diag_plus_gue", seed_h0=7)
    h.plan(mode, k=k)
    tol = 1e-13 if dtype == "c128" else 1e-7
    out, K = h.chebyshev_scan(to_dev(Psi), t, -5.2, 5.2, tol, lambdas=lam)
    out = out.cpu().numpy().astype(np.complex128)
    V = oracle.materialize(D, 8)
    h0 = oracle.h0_diagonal(D, 7)
    assert K == oracle.chebyshev_n_terms(5.2 * t, tol)
    for v in range(k):
        Hv = np.diag(h0) + lam[v] * V
        w, U = np.linalg.eigh(Hv)
        assert w[0] > -5.2 and w[-1] < 5.2
        psi_v = Psi[:, v].astype(np.complex128)
        exact = U @ (np.exp(-1j * w * t) * (U.conj().T @ psi_v))
        bound = 1e-11 if dtype == "c128" else 1e-4
        assert np.linalg.norm(out[:, v] - exact) <= bound * np.linalg.norm(psi_v), v
        if dtype == "c128":
            ref, _ = oracle.chebyshev_propagate(lambda x: Hv @ x, psi_v, t, -5.2, 5.2, tol)
            assert np.linalg.norm(out[:, v] - ref) <= 1e-11
    h.destroy()
