"""GPU parity of externally stored blocks (MFH_SRC_EXTERNAL, mfh_set_block; Eq. 10): a dense
operator held by the caller is loaded block by block into the HBM cache once and applied by the cached kernels,
against oracle/external.py (the block loop over the same array)."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import dense_matrix, make_psi

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-11, "c64": 1e-4}


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def upload(h, H, B, store, dtype, device_blocks=False):
    want = np.complex128 if dtype == "c128" else np.complex64
    for (n, m) in oracle.stored_blocks(H.shape[0] // B, store):
        blk = np.ascontiguousarray(H[n * B:(n + 1) * B, m * B:(m + 1) * B].astype(want))
        h.set_block(n, m, to_dev(blk) if device_blocks else blk)


@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("store,herm", [("full", True), ("full", False), ("pairs", True)])
@pytest.mark.parametrize("k", [1, 4])
def test_external_operator_vs_oracle(dtype, store, herm, k):
    if store == "pairs" and k > 1 and dtype == "c128":
        pytest.skip("the k-vector pair cache is the complex64 tensor-core kernel's (transposed second read)")
    D, B = 1024, 128
    H = dense_matrix(D, 11, hermitian=herm)
    if dtype == "c64":
        H = H.astype(np.complex64).astype(np.complex128)             # both sides use the rounded operator
    Psi = make_psi(D, 12, k=k, dtype=dtype)
    h = mfh.Hamiltonian(D, B, 0, dtype, kind="external", lam=1.5)
    plan = h.plan(store, k=k)
    assert plan["chosen"]["mode"] == store and plan["chosen"]["cached_fraction"] == 1.0
    with pytest.raises(mfh.MfhError) as e:                            # nothing uploaded yet
        h.apply(to_dev(Psi))
    assert e.value.code == mfh.MFH_ERR_BAD_STATE
    upload(h, H, B, store, dtype, device_blocks=(k == 1))
    Phi = h.apply(to_dev(Psi)).cpu().numpy().reshape(D, k)
    ref = 1.5 * oracle.block_apply(H, B, Psi.reshape(D, k), store)
    for v in range(k):
        assert np.linalg.norm(Phi[:, v] - ref[:, v]) <= TOL[dtype] * np.linalg.norm(ref[:, v]), v
    h.destroy()


def test_block_update_chebyshev_and_errors():
    D, B = 512, 128
    H = dense_matrix(D, 13)
    psi = make_psi(D, 14)
    h = mfh.Hamiltonian(D, B, 0, "c128", kind="external")
    for bad in ("procedural", "partial"):
        with pytest.raises(mfh.MfhError) as e:
            h.plan(bad)
        assert e.value.code == mfh.MFH_ERR_INVALID_ARG
    h.plan("pairs")
    with pytest.raises(mfh.MfhError) as e:
        h.set_block(2, 1, H[2 * B:3 * B, B:2 * B])                    # not canonical in the pair cache
    assert e.value.code == mfh.MFH_ERR_INVALID_ARG
    upload(h, H, B, "pairs", "c128")
    w, U = np.linalg.eigh(H)
    out, K = h.chebyshev(to_dev(psi), 3.0, w[0] - 0.05, w[-1] + 0.05, 1e-13)
    exact = U @ (np.exp(-3.0j * w) * (U.conj().T @ psi))
    assert np.linalg.norm(out.cpu().numpy() - exact) <= 1e-11
    # a block set again replaces the old one (time-dependent operators)
    H2 = H.copy()
    H2[:B, :B] = 2.0 * H[:B, :B]
    h.set_block(0, 0, np.ascontiguousarray(H2[:B, :B]))
    phi = h.apply(to_dev(psi)).cpu().numpy()
    assert np.linalg.norm(phi - H2 @ psi) <= 1e-11 * np.linalg.norm(H2 @ psi)
    g = mfh.Hamiltonian(D, B, 1, "c128")
    g.plan("full")
    with pytest.raises(mfh.MfhError) as e:
        g.set_block(0, 0, H[:B, :B])                                  # not an external handle
    assert e.value.code == mfh.MFH_ERR_INVALID_ARG
    h.destroy()
    g.destroy()
