"""GPU parity at BASELINE.json's full sizes (C2..C5), in the launch configuration bench.py times,
on sampled output rows the oracle computes one by one (a full oracle apply of C4 is ~6000
core-seconds), plus properties that hold at any size; and the Chebyshev propagator against the
step-by-step oracle at reduced D and by norm conservation / time reversal at full D."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import CONFIGS, lambda_grid, make_psi, sample_rows

pytestmark = pytest.mark.gpu


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def free_bytes():
    import torch
    return torch.cuda.mem_get_info()[0]


def test_c2_full_cache_sampled_rows_and_cached_equals_procedural():
    import torch
    c = CONFIGS["C2"]
    D, B = c["D"], c["B"]
    if free_bytes() < 75e9:
        pytest.skip("needs 68.7 GB of free HBM")
    psi = make_psi(D, c["psi_seed"])
    h = mfh.Hamiltonian(D, B, c["seed"], "c128")
    plan = h.plan("full", n_applies_hint=100)
    assert plan["chosen"]["mode"] == "full" and plan["chosen"]["cache_bytes"] == D * D * 16
    d_psi = to_dev(psi)
    phi_first = h.apply(d_psi).clone()
    for _ in range(5):
        phi = h.apply(d_psi)
    assert torch.equal(phi, phi_first)                     # repeated applies: bit-identical
    phi = phi.cpu().numpy()
    h.destroy()
    rows = sample_rows(D, 250)
    ref = oracle.apply(D, B, c["seed"], psi, rows=rows)
    assert rel_l2(phi[rows], ref) <= 1e-11
    assert abs(np.linalg.norm(phi) ** 2 - 1.0) < 0.05      # ||H psi||^2 = 1 + O(D^-1/2) for this GUE
    hp = mfh.Hamiltonian(D, B, c["seed"], "c128")
    hp.plan("procedural")
    phi_p = hp.apply(d_psi).cpu().numpy()
    assert rel_l2(phi, phi_p) <= 1e-13                      # caching is not an approximation


def test_c2_pair_cache_sampled_rows():
    # NEXT-1: the same operator from half the bytes (34.9 GB instead of 68.7 GB)
    c = CONFIGS["C2"]
    D, B = c["D"], c["B"]
    if free_bytes() < 40e9:
        pytest.skip("needs 35 GB of free HBM")
    psi = make_psi(D, c["psi_seed"])
    h = mfh.Hamiltonian(D, B, c["seed"], "c128")
    plan = h.plan("pairs", n_applies_hint=100)
    N = D // B
    assert plan["chosen"]["mode"] == "pairs" and plan["chosen"]["cache_bytes"] == N * (N + 1) // 2 * B * B * 16
    phi = h.apply(to_dev(psi)).cpu().numpy()
    h.destroy()
    rows = sample_rows(D, 250)
    ref = oracle.apply(D, B, c["seed"], psi, rows=rows)
    assert rel_l2(phi[rows], ref) <= 1e-11


def test_c3_scan_sampled_rows():
    c = CONFIGS["C3"]
    D, B, k = c["D"], c["B"], c["k"]
    Psi = make_psi(D, c["psi_seed"], k=k, dtype="c64")
    lam = lambda_grid(k)
    h = mfh.Hamiltonian(D, B, c["seed"], "c64", kind="diag_plus_gue", seed_h0=c["seed_h0"])
    h.plan("procedural", k=k)
    Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
    rows = sample_rows(D, 500)
    ref = oracle.apply_scan(D, B, c["seed"], c["seed_h0"], lam, Psi, rows=rows)
    for v in range(k):
        assert rel_l2(Phi[rows, v], ref[:, v]) <= 1e-4, v
    h0 = oracle.h0_diagonal(D, c["seed_h0"])
    assert rel_l2(Phi[:, 0], h0 * Psi[:, 0].astype(np.complex128)) <= 2e-7


def test_c4_procedural_sampled_rows():
    c = CONFIGS["C4"]
    D, B = c["D"], c["B"]
    psi = make_psi(D, c["psi_seed"])
    h = mfh.Hamiltonian(D, B, c["seed"], "c128")
    plan = h.plan("procedural", n_applies_hint=10)
    assert plan["chosen"]["mode"] == "procedural" and plan["dense_bytes"] == D * D * 16
    phi = h.apply(to_dev(psi)).cpu().numpy()
    rows = sample_rows(D, 120)
    ref = oracle.apply(D, B, c["seed"], psi, rows=rows)
    assert rel_l2(phi[rows], ref) <= 1e-11
    assert abs(np.linalg.norm(phi) ** 2 - 1.0) < 0.05


def test_c5_partial_cache_apply_and_chebyshev_norm():
    import torch
    c = CONFIGS["C5"]
    D, B = c["D"], c["B"]
    if free_bytes() < 160e9:
        pytest.skip("needs ~150 GB of free HBM")
    psi = make_psi(D, c["psi_seed"])
    h = mfh.Hamiltonian(D, B, c["seed"], "c128")
    plan = h.plan("partial", n_applies_hint=151, hbm_budget_bytes=int(c["hbm_budget"]))
    ch = plan["chosen"]
    assert ch["mode"] == "partial" and 0.9 * 150e9 < ch["total_bytes"] <= 150e9
    d_psi = to_dev(psi)
    phi = h.apply(d_psi).cpu().numpy()
    rows = sample_rows(D, 120)
    ref = oracle.apply(D, B, c["seed"], psi, rows=rows)
    assert rel_l2(phi[rows], ref) <= 1e-11
    out, K = h.chebyshev(d_psi, c["t"], c["e_min"], c["e_max"], c["tol"])
    assert K == 152 == oracle.chebyshev_n_terms(2.1 * c["t"], c["tol"])
    nrm = float(torch.linalg.vector_norm(out).item())
    assert abs(nrm - 1.0) <= 1e-10                          # BASELINE.json configs[4]
    back, _ = h.chebyshev(out, -c["t"], c["e_min"], c["e_max"], c["tol"])
    assert rel_l2(back.cpu().numpy(), psi) <= 1e-10         # time reversal (Eq. 40 unitarity)


@pytest.mark.parametrize("D,B,mode,budget", [(1024, 256, "procedural", 0), (2048, 512, "partial", 40e6),
                                             (8192, 1024, "full", 0)])
def test_chebyshev_vs_oracle_reduced_size(D, B, mode, budget):
    import torch
    t, tol, e0, e1 = 50.0, 1e-14, -2.1, 2.1
    psi = make_psi(D, 99)
    h = mfh.Hamiltonian(D, B, 21, "c128")
    h.plan(mode, hbm_budget_bytes=int(budget))
    out, K = h.chebyshev(to_dev(psi), t, e0, e1, tol)
    out = out.cpu().numpy()
    H = oracle.materialize(D, 21)
    ref, K_ref = oracle.chebyshev_propagate(lambda v: H @ v, psi, t, e0, e1, tol)
    assert K == K_ref == 152
    assert rel_l2(out, ref) <= 1e-11
    assert abs(np.linalg.norm(out) - 1.0) <= 1e-10


def test_chebyshev_t0_is_identity_and_bad_args():
    D, B = 1024, 256
    psi = make_psi(D, 99)
    h = mfh.Hamiltonian(D, B, 21, "c128")
    h.plan("procedural")
    out, K = h.chebyshev(to_dev(psi), 0.0, -2.1, 2.1, 1e-14)
    assert K == 1 and rel_l2(out.cpu().numpy(), psi) <= 1e-15
    with pytest.raises(mfh.MfhError) as e:
        h.chebyshev(to_dev(psi), 1.0, 2.1, -2.1, 1e-14)
    assert e.value.code == mfh.MFH_ERR_INVALID_ARG
    with pytest.raises(mfh.MfhError):
        h.chebyshev(to_dev(psi), float("inf"), -2.1, 2.1, 1e-14)


def test_chebyshev_shifted_asymmetric_bounds():
    # c != 0 exercises the -c q term of H~ and the e^{-ict} phase
    D, B = 1024, 256
    psi = make_psi(D, 5)
    h = mfh.Hamiltonian(D, B, 21, "c128")
    h.plan("procedural")
    out, K = h.chebyshev(to_dev(psi), 7.5, -2.2, 2.6, 1e-13)
    H = oracle.materialize(D, 21)
    ref, K_ref = oracle.chebyshev_propagate(lambda v: H @ v, psi, 7.5, -2.2, 2.6, 1e-13)
    assert K == K_ref
    assert rel_l2(out.cpu().numpy(), ref) <= 1e-11


def test_c3_scan_from_cached_blocks_sampled_rows():
    """C3's operator cached (8.6 GB complex64 -> tensor-core kernel; 17.2 GB complex128 -> FP64 kernel)."""
    c = CONFIGS["C3"]
    D, B, k = c["D"], c["B"], c["k"]
    lam = lambda_grid(k)
    rows = sample_rows(D, 200)
    for dtype, tol in (("c64", 1e-4), ("c128", 1e-11)):
        Psi = make_psi(D, c["psi_seed"], k=k, dtype=dtype)
        h = mfh.Hamiltonian(D, B, c["seed"], dtype, kind="diag_plus_gue", seed_h0=c["seed_h0"])
        plan = h.plan("full", k=k)
        assert plan["chosen"]["cache_bytes"] == D * D * (8 if dtype == "c64" else 16)
        Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
        ref = oracle.apply_scan(D, B, c["seed"], c["seed_h0"], lam, Psi, rows=rows)
        for v in range(k):
            assert rel_l2(Phi[rows, v], ref[:, v]) <= tol, (dtype, v)
        h.destroy()


def test_c4_partitioned_over_8_ranks():
    """NEXT-4 at C4's size, one rank after the other on this GPU: the eight pair-set contributions add up to the
    single-GPU apply (partition invariance, "does not change the Hamiltonian or omit any block
    products"), and a row-slab rank reproduces its rows of the oracle and leaves the others untouched."""
    import torch
    c = CONFIGS["C4"]
    D, B = c["D"], c["B"]
    psi_np = make_psi(D, c["psi_seed"])
    psi = to_dev(psi_np)
    h = mfh.Hamiltonian(D, B, c["seed"], "c128")
    h.plan("procedural")
    full = h.apply(psi).clone()
    h.destroy()
    total = torch.zeros_like(full)
    for r in range(8):
        hr = mfh.Hamiltonian(D, B, c["seed"], "c128")
        hr.set_partition(r, 8, "pairs")
        hr.plan("procedural")
        total += hr.apply(psi)
        hr.destroy()
    assert float(torch.linalg.vector_norm(total - full) / torch.linalg.vector_norm(full)) <= 1e-13
    hr = mfh.Hamiltonian(D, B, c["seed"], "c128")
    hr.set_partition(5, 8, "rows")
    hr.plan("procedural")
    lo, cnt = hr.partition_rows()
    assert (lo, cnt) == (5 * D // 8, D // 8)
    phi = torch.full_like(full, 3.0 - 4.0j)
    hr.apply(psi, phi)
    got = phi.cpu().numpy()
    rows = lo + sample_rows(cnt, 60)
    ref = oracle.apply(D, B, c["seed"], psi_np, rows=rows)
    assert rel_l2(got[rows], ref) <= 1e-11
    assert np.all(got[:lo] == 3.0 - 4.0j) and np.all(got[lo + cnt:] == 3.0 - 4.0j)
    assert rel_l2(got[lo:lo + cnt], full.cpu().numpy()[lo:lo + cnt]) <= 1e-13
    hr.destroy()
