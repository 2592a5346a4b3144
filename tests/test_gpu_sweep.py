"""Seeded sweep of small shapes through every mode of the CUDA path against the oracle: odd block counts, a
single block, the smallest block, odd numbers of cached block diagonals, every k, empty ranks of a partitioned
job.  Each case is tiny (D <= 1152); the point is the corner cases of the planner tables and the kernels' tails."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import lambda_grid, make_psi

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-11, "c64": 1e-4}


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def _cases():
    rng = np.random.default_rng(20260631)
    shapes = [(32, 32), (64, 32), (96, 32), (160, 32), (128, 128), (384, 128), (640, 128), (1152, 128), (192, 64),
              (448, 64), (768, 256), (288, 96), (480, 96)]
    out = []
    for (D, B) in shapes:
        for dtype in ("c128", "c64"):
            for mode in ("procedural", "partial", "full", "pairs"):
                k = int(rng.choice([1, 1, 1, 2, 3, 5, 8, 13, 16]))
                if mode == "pairs" and k > 1 and not (dtype == "c64" and B % 128 == 0):
                    k = 1                                      # k-vector pair caches: complex64, B % 128 == 0 only
                if mode == "pairs" and k == 1 and dtype == "c64" and B % 64:
                    continue
                if k > 1 and mode in ("partial", "full") and B % 128:
                    continue                                   # cached k-vector kernels need B % 128 == 0
                frac = float(rng.choice([0.2, 0.45, 0.7]))
                out.append((D, B, dtype, mode, k, frac, int(rng.integers(1, 2**31))))
    return out


@pytest.mark.parametrize("D,B,dtype,mode,k,frac,seed", _cases())
def test_small_shape_sweep(D, B, dtype, mode, k, frac, seed):
    cb = 16 if dtype == "c128" else 8
    n_blk = D // B
    if mode == "partial" and n_blk < 2:
        pytest.skip("a single block has no partial cache")
    Psi = make_psi(D, seed % 1000, k=k, dtype=dtype)
    lam = lambda_grid(k) + 0.3
    h = mfh.Hamiltonian(D, B, seed, dtype, kind="diag_plus_gue", seed_h0=seed + 1)
    budget = 0
    if mode == "partial":                                      # room for about `frac` of the blocks plus the workspace
        budget = int(frac * D * D * cb + 64 * D * k * cb + (1 << 20))
    try:
        plan = h.plan(mode, k=k, hbm_budget_bytes=budget)
    except mfh.MfhError as e:
        assert e.code == mfh.MFH_ERR_OUT_OF_MEMORY and mode == "partial"    # nothing fits the tiny budget
        return
    Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy().reshape(D, k)
    ref = oracle.apply_scan(D, B, seed, seed + 1, lam, Psi.reshape(D, k))
    for v in range(k):
        err = np.linalg.norm(Phi[:, v] - ref[:, v]) / np.linalg.norm(ref[:, v])
        assert err <= TOL[dtype], (plan["chosen"], v, err)
    h.destroy()


@pytest.mark.parametrize("scheme", ["rows", "pairs"])
@pytest.mark.parametrize("D,B,world", [(96, 32, 5), (128, 128, 2), (320, 64, 3), (640, 128, 4)])
def test_partition_with_empty_and_ragged_ranks(scheme, D, B, world):
    """More ranks than block rows / pairs: some ranks own nothing and must contribute exactly zero."""
    import torch
    seed = 77
    psi = make_psi(D, 5)
    full = oracle.apply(D, B, seed, psi)
    total = np.zeros(D, dtype=np.complex128)
    for r in range(world):
        h = mfh.Hamiltonian(D, B, seed, "c128")
        h.set_partition(r, world, scheme)
        h.plan("procedural")
        phi = torch.zeros(D, dtype=torch.complex128, device="cuda")
        h.apply(to_dev(psi), phi)
        got = phi.cpu().numpy()
        ref = oracle.apply_partition(D, B, seed, psi, r, world, scheme)
        assert np.linalg.norm(got - ref) <= 1e-11 * np.linalg.norm(full), (r, scheme)
        total += got
        h.destroy()
    assert np.linalg.norm(total - full) <= 1e-11 * np.linalg.norm(full)
