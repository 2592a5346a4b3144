"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Tolerances (BASELINE.json north_star): Philox words bit-exact; relative L2
||phi_gpu - phi_cpu|| / ||phi_cpu|| <= 1e-11 for complex128, <= 1e-4 for complex64 (per column).
"""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import CONFIGS, lambda_grid, make_psi

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-11, "c64": 1e-4}


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def gpu_apply(D, B, seed, psi, dtype="c128", mode="procedural", k=1, budget=0, **kw):
    h = mfh.Hamiltonian(D, B, seed, dtype, **kw)
    plan = h.plan(mode, k=k, hbm_budget_bytes=budget)
    phi = h.apply(to_dev(psi)).cpu().numpy()
    return phi, plan, h


# ---- generator ------------------------------------------------------------------------------

def _philox_gpu(seed, stream, i, j):
    import torch
    w = mfh.debug_philox(seed, stream, to_dev(i.astype(np.uint32).view(np.int32)),
                         to_dev(j.astype(np.uint32).view(np.int32)))
    torch.cuda.synchronize()
    return w.cpu().numpy().view(np.uint32)


def test_philox_words_bit_exact_block00_of_c1():
    a = np.arange(512, dtype=np.uint32)
    i, j = [x.ravel() for x in np.meshgrid(a, a, indexing="ij")]
    assert np.array_equal(_philox_gpu(1234, 0, i, j), oracle.philox_pairs(1234, 0, i, j))


def test_philox_words_bit_exact_random_pairs_and_corners():
    rng = np.random.default_rng(5)
    i = rng.integers(0, 262144, size=1_000_000).astype(np.uint32)
    j = rng.integers(0, 262144, size=1_000_000).astype(np.uint32)
    D = 262144
    i[:4] = [0, 0, D - 1, D - 1]
    j[:4] = [0, D - 1, 0, D - 1]
    for seed, stream in [(1234, 0), (7, 1), (2**40 + 3, 0)]:
        assert np.array_equal(_philox_gpu(seed, stream, i, j), oracle.philox_pairs(seed, stream, i, j))


def test_philox_empty_input():
    import torch
    e = torch.empty(0, dtype=torch.int32, device="cuda")
    assert mfh.debug_philox(1, 0, e, e).shape == (0, 4)


# c128 tolerance: DESIGN.md 6.2 "Generator arithmetic" (log1p remainder 6e-15, table rounding)
@pytest.mark.parametrize("dtype,tol", [("c128", 3e-14), ("c64", 3e-6)])
@pytest.mark.parametrize("n,m", [(0, 0), (0, 3), (3, 0), (7, 7)])
def test_materialized_block_matches_oracle_entries(dtype, tol, n, m):
    D, B = 4096, 512
    h = mfh.Hamiltonian(D, B, 1234, dtype)
    blk = h.materialize_block(n, m, B).cpu().numpy().astype(np.complex128)
    ref = oracle.materialize(D, 1234, n * B, B, m * B, B)
    # entries are O(1/sqrt(D)); absolute error relative to that scale
    assert np.abs(blk - ref).max() * np.sqrt(D) < tol * 50
    assert rel_l2(blk, ref) < tol
    if n == m:
        assert np.all(blk.imag.diagonal() == 0.0)
        assert np.array_equal(blk, blk.conj().T)          # bit-exact Hermiticity


def test_h0_diagonal_matches_oracle():
    h = mfh.Hamiltonian(32768, 1024, 8, "c128", kind="diag_plus_gue", seed_h0=7)
    assert np.array_equal(h.h0().cpu().numpy(), oracle.h0_diagonal(32768, 7))


# ---- C1: procedural apply vs oracle and vs explicit dense matmul ----------------------------

def test_c1_procedural_vs_oracle_and_dense():
    c = CONFIGS["C1"]
    psi = make_psi(c["D"], c["psi_seed"])
    phi, plan, h = gpu_apply(c["D"], c["B"], c["seed"], psi)
    assert plan["chosen"]["mode"] == "procedural"
    ref = oracle.apply(c["D"], c["B"], c["seed"], psi)
    assert rel_l2(phi, ref) <= TOL["c128"]
    H = oracle.materialize(c["D"], c["seed"])
    assert rel_l2(phi, H @ psi) <= TOL["c128"]


@pytest.mark.parametrize("mode,budget", [("procedural", 0), ("full", 0), ("partial", 12e6),
                                         ("partial", 30e6), ("partial", 60e6), ("pairs", 0), ("pairs", 12e6),
                                         ("pairs", 20e6), ("pairs", 30e6)])
@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_modes_agree_with_oracle(mode, budget, dtype):
    D, B = 2048, 256          # 8x8 blocks of 1 MiB (c128): budgets cache ~1..6 blocks per row
    psi = make_psi(D, 3, dtype=dtype)
    if dtype == "c64":
        budget = budget / 2
    phi, plan, h = gpu_apply(D, B, 42, psi, dtype=dtype, mode=mode, budget=int(budget))
    assert plan["chosen"]["mode"] == mode
    ref = oracle.apply(D, B, 42, psi)
    assert rel_l2(phi, ref) <= TOL[dtype]


@pytest.mark.parametrize("D,B", [(32, 32), (96, 32), (160, 32), (1024, 1024), (4096, 4096), (3072, 1024),
                                 (2048, 64), (4096, 128), (1536, 512), (8192, 2048)])
def test_partition_invariance_and_ragged_shapes(D, B):
    # the operator must not depend on the partition
    psi = make_psi(D, 17)
    phi, _, _ = gpu_apply(D, B, 1234, psi)
    ref = oracle.apply(D, B, 1234, psi)
    assert rel_l2(phi, ref) <= TOL["c128"]


@pytest.mark.parametrize("D,B", [(32, 32), (96, 32), (1024, 1024), (3072, 1024), (2048, 64), (1536, 512)])
@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_pair_cache_ragged_shapes(D, B, dtype):
    # Hermitian pair cache: one stored block serves (n,m) and (m,n); odd and even N_blk,
    # a single block, the smallest block size of each dtype
    if dtype == "c64" and B % 64:
        pytest.skip("c64 pair cache needs B % 64 == 0 (two entries per 128-bit load)")
    psi = make_psi(D, 23, dtype=dtype)
    phi, plan, h = gpu_apply(D, B, 77, psi, dtype=dtype, mode="pairs")
    ch = plan["chosen"]
    N = D // B
    assert ch["mode"] == "pairs" and ch["cached_blocks"] == N * (N + 1) // 2 and ch["cached_fraction"] == 1.0
    assert rel_l2(phi, oracle.apply(D, B, 77, psi)) <= TOL[dtype]


def test_apply_is_deterministic_and_repeatable():
    import torch
    D, B = 4096, 512
    psi = to_dev(make_psi(D, 1))
    for mode, budget in [("procedural", 0), ("partial", int(150e6)), ("pairs", 0), ("pairs", int(100e6))]:
        h = mfh.Hamiltonian(D, B, 9, "c128")
        h.plan(mode, hbm_budget_bytes=budget)
        a = h.apply(psi).clone()
        for _ in range(3):
            b = h.apply(psi)
            assert torch.equal(a, b)                      # no atomics in the complex128 path


def test_hermiticity_on_gpu():
    D, B = 4096, 512
    a, b = make_psi(D, 1), make_psi(D, 2)
    h = mfh.Hamiltonian(D, B, 77, "c128")
    h.plan("procedural")
    Ha = h.apply(to_dev(a)).cpu().numpy()
    Hb = h.apply(to_dev(b)).cpu().numpy()
    assert abs(np.vdot(a, Hb) - np.conj(np.vdot(b, Ha))) < 1e-13


@pytest.mark.parametrize("mode,budget", [("procedural", 0), ("full", 0), ("partial", 30e6), ("pairs", 0), ("pairs", 20e6)])
@pytest.mark.parametrize("dtype", ["c128", "c64"])
def test_h0_plus_lambda_v_single_vector_all_modes(mode, budget, dtype):
    # H = diag(h0) + lambda V with one vector: the epilogue of the reduce kernel on top of every cache mode
    # (complex128 partial = the overlapped kernel, complex64 partial = cached + fused kernels back to back)
    D, B, lam = 2048, 256, 0.7
    psi = make_psi(D, 6, dtype=dtype)
    if dtype == "c64":
        budget = budget / 2
    phi, plan, h = gpu_apply(D, B, 8, psi, dtype=dtype, mode=mode, budget=int(budget), kind="diag_plus_gue",
                             lam=lam, seed_h0=7)
    assert plan["chosen"]["mode"] == mode
    ref = oracle.apply_scan(D, B, 8, 7, [lam], psi.reshape(D, 1))[:, 0]
    assert rel_l2(phi, ref) <= TOL[dtype]


def test_lambda_scales_single_vector():
    D, B = 1024, 256
    psi = make_psi(D, 4)
    phi, _, _ = gpu_apply(D, B, 5, psi, lam=0.37)
    assert rel_l2(phi, 0.37 * oracle.apply(D, B, 5, psi)) <= TOL["c128"]


# ---- multi-vector / coupling scan (C3 shape) -------------------------------------------------

@pytest.mark.parametrize("dtype,k", [("c64", 16), ("c64", 5), ("c128", 4), ("c128", 16), ("c64", 2)])
def test_scan_multi_vector_vs_oracle(dtype, k):
    D, B = 2048, 256
    Psi = make_psi(D, 9, k=k, dtype=dtype)
    lam = lambda_grid(k)
    h = mfh.Hamiltonian(D, B, 8, dtype, kind="diag_plus_gue", seed_h0=7)
    h.plan("procedural", k=k)
    Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
    ref = oracle.apply_scan(D, B, 8, 7, lam, Psi)
    for v in range(k):
        assert rel_l2(Phi[:, v], ref[:, v]) <= TOL[dtype], v
    # lambda_0 = 0: column 0 is the textbook special case h0 (.) psi_0
    h0 = oracle.h0_diagonal(D, 7)
    assert rel_l2(Phi[:, 0], h0 * Psi[:, 0].astype(np.complex128)) <= (1e-15 if dtype == "c128" else 2e-7)


@pytest.mark.parametrize("D,B", [(128, 128), (1024, 128), (3072, 1024), (960, 96), (2048, 64)])
@pytest.mark.parametrize("k", [16, 3])
def test_scan_c64_tensor_core_and_cuda_core_shapes(D, B, k):
    # complex64 k-vector path: B % 128 == 0 runs the tcgen05 kernel (3xTF32, A operand in TMEM),
    # other block sizes the CUDA-core kernel; a single block (all entries from the general rule),
    # blocks above and below the diagonal, ragged N_blk
    Psi = make_psi(D, 31, k=k, dtype="c64")
    lam = 0.5 + lambda_grid(k)
    h = mfh.Hamiltonian(D, B, 8, "c64", kind="diag_plus_gue", seed_h0=7)
    h.plan("procedural", k=k)
    Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
    ref = oracle.apply_scan(D, B, 8, 7, lam, Psi)
    for v in range(k):
        assert rel_l2(Phi[:, v], ref[:, v]) <= TOL["c64"], v


def test_scan_c64_two_sided_tensor_core_kernels_and_their_fallbacks():
    """complex64 k-vector plans use the Hermitian structure on the tensor cores (Eq. 11): a block
    pair whose two positions are generated is generated ONCE (pairs_tc_kernel<false>), a stored pair of a pair cache is
    read ONCE (pairs_tc_kernel<true>, unit-image layout); both need B/128 extra partial slots per block row and fall
    back to the one-sided kernels when those do not fit the budget.  Same oracle, same tolerance, every path."""
    D, B, k = 2048, 256, 16
    nb = D // B
    Psi = make_psi(D, 17, k=k, dtype="c64")
    lam = 0.25 + lambda_grid(k)
    ref = oracle.apply_scan(D, B, 8, 7, lam, Psi)
    # mode, budget, generated pairs served two-sided, stored pairs served two-sided
    cases = [("procedural", 0, nb * (nb - 1) // 2, 0),          # every off-diagonal pair generated once
             ("procedural", 6_000_000, 0, 0),                   # the column-side slots do not fit: one-sided generation
             ("pairs", 0, 0, nb * (nb - 1) // 2),               # every stored off-diagonal pair read once
             ("pairs", 14_000_000, 0, 0)]                       # tight budget: as many stored pairs as fit WITHOUT the extra
                                                                # slots (transposed second read), the rest generated one-sided
    for mode, budget, n_gen, n_stored in cases:
        h = mfh.Hamiltonian(D, B, 8, "c64", kind="diag_plus_gue", seed_h0=7)
        h.plan(mode, k=k, hbm_budget_bytes=budget)
        gp = h.get_plan()
        assert (gp["two_sided_pairs"], gp["two_sided_stored_pairs"]) == (n_gen, n_stored), (mode, budget, gp)
        if mode == "pairs" and budget:
            assert 0 < gp["cached_blocks"] < nb * (nb + 1) // 2, gp
        h.debug_poison()                                          # a slot that is read but not written turns the result into NaN
        Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
        for v in range(k):
            assert rel_l2(Phi[:, v], ref[:, v]) <= TOL["c64"], (mode, budget, v)
        h.destroy()


@pytest.mark.parametrize("D,B,k", [(4096, 2048, 16), (8192, 4096, 7), (768, 384, 16), (3072, 1536, 2)])
@pytest.mark.parametrize("mode", ["procedural", "pairs"])
def test_scan_c64_two_sided_kernels_block_sizes(D, B, k, mode):
    """The two-sided tensor-core kernels build the next item's psi operand a few rows per unit (B / 32 units per item):
    one row pair per unit from B = 2048 (the block size the measured planner picks for C3's operator), two up to
    B = 1024, more below; B = 384 and 1536 are multiples of 128 that are not powers of two."""
    Psi = make_psi(D, 23, k=k, dtype="c64")
    lam = 0.5 + lambda_grid(k)
    h = mfh.Hamiltonian(D, B, 8, "c64", kind="diag_plus_gue", seed_h0=7)
    h.plan(mode, k=k)
    gp = h.get_plan()
    assert gp["two_sided_pairs" if mode == "procedural" else "two_sided_stored_pairs"] == (D // B) * (D // B - 1) // 2
    h.debug_poison()
    Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
    ref = oracle.apply_scan(D, B, 8, 7, lam, Psi)
    for v in range(k):
        assert rel_l2(Phi[:, v], ref[:, v]) <= TOL["c64"], v
    h.destroy()


@pytest.mark.parametrize("mode,budget", [("full", 0), ("partial", 12e6), ("partial", 24e6)])
@pytest.mark.parametrize("dtype,k", [("c64", 16), ("c64", 5), ("c128", 16), ("c128", 8), ("c128", 3), ("c128", 2)])
def test_scan_cached_blocks_k_vectors(mode, budget, dtype, k):
    # cached k-vector path: each stored V block is read once for all k vectors (complex64: TMA -> TMEM ->
    # tcgen05; complex128: cp.async staging -> FP64 CUDA cores), alone and mixed with generated blocks
    D, B = 2048, 256          # 8x8 blocks of 512 KiB (c64) / 1 MiB (c128)
    Psi = make_psi(D, 13, k=k, dtype=dtype)
    lam = 0.25 + lambda_grid(k)
    h = mfh.Hamiltonian(D, B, 8, dtype, kind="diag_plus_gue", seed_h0=7)
    plan = h.plan(mode, k=k, hbm_budget_bytes=int(budget * (2 if dtype == "c128" else 1)))
    assert plan["chosen"]["mode"] == mode
    Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
    ref = oracle.apply_scan(D, B, 8, 7, lam, Psi)
    for v in range(k):
        assert rel_l2(Phi[:, v], ref[:, v]) <= TOL[dtype], v


def test_scan_c128_cached_single_block_and_min_block():
    # one 128 x 128 block (every entry from the general rule) and the smallest supported block size
    for D, B, k in [(128, 128, 16), (1024, 128, 7)]:
        Psi = make_psi(D, 17, k=k)
        lam = lambda_grid(k)
        h = mfh.Hamiltonian(D, B, 8, "c128", kind="diag_plus_gue", seed_h0=7)
        h.plan("full", k=k)
        Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
        ref = oracle.apply_scan(D, B, 8, 7, lam, Psi)
        for v in range(k):
            assert rel_l2(Phi[:, v], ref[:, v]) <= TOL["c128"], (D, v)


def test_multi_vector_equals_single_vector_applies():
    D, B, k = 1024, 256, 4
    Psi = make_psi(D, 21, k=k)
    h = mfh.Hamiltonian(D, B, 8, "c128")
    h.plan("procedural", k=k)
    Phi = h.apply(to_dev(Psi)).cpu().numpy()
    h1 = mfh.Hamiltonian(D, B, 8, "c128")
    h1.plan("procedural", k=1)
    for v in range(k):
        one = h1.apply(to_dev(Psi[:, v].copy())).cpu().numpy()
        assert rel_l2(Phi[:, v], one) <= 1e-13


# ---- planner on the device -------------------------------------------------------------------

def test_measured_planner_commits_a_working_plan():
    D = 4096
    psi = make_psi(D, 2)
    h = mfh.Hamiltonian(D, 0, 1234, "c128")
    rec = h.plan("auto", n_applies_hint=50, measure=True)
    assert rec["planner"] == "measured" and rec["chosen"]["measured_apply_s"] > 0
    timed = [c for c in rec["candidates"] if c["measured_apply_s"] > 0]
    assert 1 <= len(timed) <= 8                            # K_bench <= 8
    B = h.get_plan()["B"]
    assert rel_l2(h.apply(to_dev(psi)).cpu().numpy(), oracle.apply(D, B, 1234, psi)) <= TOL["c128"]


def test_plan_k_mismatch_and_replan():
    import torch
    D = 1024
    h = mfh.Hamiltonian(D, 256, 1, "c128")
    h.plan("procedural", k=2)
    h.k = 1
    with pytest.raises(mfh.MfhError) as e:
        h.apply(torch.zeros(D, dtype=torch.complex128, device="cuda"))
    assert e.value.code == mfh.MFH_ERR_INVALID_ARG
    h.plan("full", k=1)                                   # re-plan is allowed
    psi = make_psi(D, 2)
    assert rel_l2(h.apply(to_dev(psi)).cpu().numpy(), oracle.apply(D, 256, 1, psi)) <= TOL["c128"]


def test_apply_host_roundtrip():
    import torch
    D, B = 2048, 256
    psi = make_psi(D, 6)
    h = mfh.Hamiltonian(D, B, 3, "c128")
    h.plan("procedural")
    ph = torch.from_numpy(psi).pin_memory()
    out = torch.empty_like(ph).pin_memory()
    h.apply_host(ph, out)
    assert rel_l2(out.numpy(), oracle.apply(D, B, 3, psi)) <= TOL["c128"]


def test_read_only_stream_probe_reports_a_plausible_hbm_rate():
    import torch
    buf = torch.ones(2 * 2**30, dtype=torch.uint8, device="cuda")       # 2 GiB, far above the 126 MB L2
    gbs = mfh.read_bandwidth(buf) / 1e9
    assert 3000.0 < gbs < 8200.0                                       # B200 HBM3e: ~8 TB/s nominal
    with pytest.raises(mfh.MfhError) as e:
        mfh.read_bandwidth(buf[:1024])
    assert e.value.code == mfh.MFH_ERR_INVALID_ARG


def test_hybrid_surrogate_planner_commits_a_working_plan():
    """Algorithm 3: rank by the surrogate trained on the shipped B200 log, time the top 3, apply."""
    import os
    from paper_2606_31598_b200 import surrogate as sur
    X, t, _ = sur.load_log(os.path.join(os.path.dirname(sur.__file__), "data", "plan_log_b200.jsonl"))
    theta, _ = sur.fit(X, t, hidden=16, epochs=2000, lr=0.01, seed=1)
    D = 8192
    h, rep = sur.hybrid_plan(theta, D, "c128", seed=1234, n_applies_hint=100, k_nn=3)
    assert len(rep["timed"]) == 3 and rep["feasible_candidates"] > 3
    assert rep["chosen"]["job_s"] == min(x["job_s"] for x in rep["timed"])
    assert all(0.2 < x["t_nn_s"] / x["measured_apply_s"] < 5.0 for x in rep["timed"])     # the ranking is informed
    psi = make_psi(D, 99)
    phi = h.apply(to_dev(psi)).cpu().numpy()
    B = h.get_plan()["B"]
    rows = np.arange(0, D, 61)
    assert rel_l2(phi[rows], oracle.apply(D, B, 1234, psi, rows=rows)) <= TOL["c128"]
    h.destroy()
