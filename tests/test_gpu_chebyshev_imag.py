"""GPU parity of the imaginary-time Chebyshev filter (mfh_chebyshev_imag, R21) against the
oracle's step-by-step series and the exact eigh filter."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import make_psi

pytestmark = pytest.mark.gpu


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("mode", ["procedural", "pairs", "partial"])
@pytest.mark.parametrize("beta", [0.2, 5.0, 40.0])
def test_filter_vs_oracle_and_eigh(mode, beta):
    D, B, seed = 2048, 256, 21
    psi = make_psi(D, 99)
    h = mfh.Hamiltonian(D, B, seed, "c128")
    h.plan(mode, hbm_budget_bytes=int(0.5 * D * D * 16) if mode == "partial" else 0)
    out, K = h.chebyshev_imag(to_dev(psi), beta, -2.2, 2.1, 1e-14)
    out = out.cpu().numpy()
    H = oracle.materialize(D, seed)
    ref, K_ref = oracle.chebyshev_imag_propagate(lambda v: H @ v, psi, beta, -2.2, 2.1, 1e-14)
    assert K == K_ref
    # the filter is a contraction: its output can be orders of magnitude below ||psi|| (beta = 40: ~1e-5), while the
    # rounding of the K-term series is absolute in ||psi||, so that is the scale of the tolerance
    assert np.linalg.norm(out - ref) <= 1e-11 * np.linalg.norm(psi)
    w, U = np.linalg.eigh(H)
    exact = U @ (np.exp(-beta * (w + 2.2)) * (U.conj().T @ psi))
    assert np.linalg.norm(out - exact) <= 1e-11 * np.linalg.norm(psi)
    h.destroy()


def test_beta_zero_identity_semigroup_and_bad_args():
    import torch
    D, B = 1024, 128
    psi = to_dev(make_psi(D, 4))
    h = mfh.Hamiltonian(D, B, 21, "c128")
    h.plan("procedural")
    o0, K0 = h.chebyshev_imag(psi, 0.0, -2.1, 2.1, 1e-14)
    assert K0 == 1 and torch.equal(o0, psi)
    a, _ = h.chebyshev_imag(psi, 1.5, -2.1, 2.1, 1e-15)
    b, _ = h.chebyshev_imag(a, 2.5, -2.1, 2.1, 1e-15)
    c, _ = h.chebyshev_imag(psi, 4.0, -2.1, 2.1, 1e-15)
    assert float(torch.linalg.vector_norm(b - c)) <= 1e-13
    for args in [(-1.0, -2.1, 2.1, 1e-14), (1.0, 2.1, -2.1, 1e-14), (1.0, -2.1, 2.1, 0.0), (1000.0, -2.1, 2.1, 1e-14),
                 (float("nan"), -2.1, 2.1, 1e-14)]:
        with pytest.raises(mfh.MfhError) as e:
            h.chebyshev_imag(psi, *args)
        assert e.value.code == mfh.MFH_ERR_INVALID_ARG
    h.destroy()


def test_c64_filter_within_the_single_precision_tolerance():
    D, B, seed, beta = 2048, 256, 21, 3.0
    psi = make_psi(D, 99, dtype="c64")
    h = mfh.Hamiltonian(D, B, seed, "c64")
    h.plan("procedural")
    out, K = h.chebyshev_imag(to_dev(psi), beta, -2.1, 2.1, 1e-7)
    H = oracle.materialize(D, seed)
    ref, K_ref = oracle.chebyshev_imag_propagate(lambda v: H @ v, psi.astype(np.complex128), beta, -2.1, 2.1, 1e-7)
    assert K == K_ref
    assert np.linalg.norm(out.cpu().numpy() - ref) <= 1e-4 * np.linalg.norm(psi)
    h.destroy()
