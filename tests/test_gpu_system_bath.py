"""GPU parity of the NEXT-3 widening: the system-bath Hamiltonian action -- two dense
bath-side operators on R = d_S state components -- against the oracle, at small size element by
element (the paper's size, 18 qubits, is covered in test_gpu_fullsize.py)."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import make_psi, small_hermitian

pytestmark = pytest.mark.gpu


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("dtype,mode,d_S", [("c64", "full", 4), ("c64", "procedural", 4), ("c64", "partial", 3),
                                            ("c128", "procedural", 4), ("c64", "full", 16), ("c128", "full", 4),
                                            ("c128", "partial", 5)])
def test_system_bath_small_vs_oracle(dtype, mode, d_S):
    d_B, B, g = 2048, 256, 0.6
    H_S, A = small_hermitian(d_S, 33), small_hermitian(d_S, 34)
    X = make_psi(d_B, 35, k=d_S, dtype=dtype)
    sb = mfh.SystemBath(d_B, d_S, B, 31, 32, H_S, A, g, dtype=dtype)
    plan = sb.plan(mode, hbm_budget_bytes=int(24e6 * (2 if dtype == "c128" else 1)) if mode == "partial" else 0)
    assert plan["n_op"] == 2 and plan["H_B"]["mode"] == mode and plan["B_1"]["mode"] == mode
    Y = sb.apply(to_dev(X)).cpu().numpy()
    ref = oracle.sb_apply(d_B, B, 31, 32, H_S, A, g, X)
    tol = 1e-11 if dtype == "c128" else 1e-4
    for s in range(d_S):
        assert rel_l2(Y[:, s], ref[:, s]) <= tol, s
    sb.destroy()


def test_system_bath_rejects_non_hermitian_system_operators():
    M = np.array([[0, 1], [2, 0]], dtype=np.complex128)
    with pytest.raises(mfh.MfhError) as e:
        mfh.SystemBath(1024, 2, 256, 1, 2, M, M.conj().T @ M, 0.1)
    assert e.value.code == mfh.MFH_ERR_INVALID_ARG
