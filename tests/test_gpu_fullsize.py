"""GPU parity at BASELINE.json's full sizes (C2..C5, the paper's 18-qubit system-bath shape), in the launch
configuration bench.py times.

Evidence per config:
  * C2 and C3: a FULL oracle apply (every output row; 15 s and ~10 s on the GPU box's 16 host threads);
  * C4, C5 (partial and pair cache), C3 from cached complex128 blocks and SB18: >= 8192 stratified rows
    (inputs.stratified_rows: every 128-row tile, every residue mod 128, i.e. every (lane, row-in-lane) position of
    the fused kernel's row tile, every block row, first and last row of every block);
  * all-row GPU-vs-GPU cross checks for the kernels that have no full oracle apply: partial-overlap vs procedural
    vs pair cache (C5), SB18 complex64 cached vs complex128 generated;
  * besides the relative L2 of north_star (1e-11 complex128, 1e-4 complex64) a PER-ELEMENT bound
    max |delta| <= 10 tol rms(ref): a single wrong row (|delta| ~ rms(ref)) fails it by ten orders of magnitude even
    where it would hide in an L2 norm over thousands of rows;
  * the Chebyshev propagator against the step-by-step oracle at reduced D and by norm conservation / time reversal
    at full D.
Oracle references are computed once per session and shared between the tests of a config."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import (CONFIGS, SYSTEM_BATH, lambda_grid, make_psi, sample_rows, small_hermitian,
                                          stratified_rows)

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-11, "c64": 1e-4}


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def check(got, ref, tol, what=""):
    """north_star's relative L2 and the per-element bound max |delta| <= 10 tol rms(ref)."""
    got = np.asarray(got, dtype=np.complex128)
    ref = np.asarray(ref, dtype=np.complex128)
    assert got.shape == ref.shape, (what, got.shape, ref.shape)
    err = rel_l2(got, ref)
    assert err <= tol, (what, "rel L2", err)
    rms = float(np.linalg.norm(ref) / np.sqrt(ref.size))
    worst = float(np.max(np.abs(got - ref)))
    assert worst <= 10.0 * tol * rms, (what, "max |delta| / rms", worst / rms, "at", int(np.argmax(np.abs(got - ref))))
    return err


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def free_bytes():
    import torch
    return torch.cuda.mem_get_info()[0]


_REF = {}


def oracle_ref(name):
    """(rows or None = all rows, reference) of a config, computed once per session."""
    if name in _REF:
        return _REF[name]
    if name == "C2":
        c = CONFIGS["C2"]
        rows, ref = None, oracle.apply(c["D"], c["B"], c["seed"], make_psi(c["D"], c["psi_seed"]))
    elif name in ("C4", "C5"):
        c = CONFIGS[name]
        rows = stratified_rows(c["D"], c["B"])
        ref = oracle.apply(c["D"], c["B"], c["seed"], make_psi(c["D"], c["psi_seed"]), rows=rows)
    elif name in ("C3", "C3-c128"):
        c = CONFIGS["C3"]
        dtype = "c64" if name == "C3" else "c128"
        Psi = make_psi(c["D"], c["psi_seed"], k=c["k"], dtype=dtype)
        rows = None if name == "C3" else stratified_rows(c["D"], c["B"])
        ref = oracle.apply_scan(c["D"], c["B"], c["seed"], c["seed_h0"], lambda_grid(c["k"]), Psi, rows=rows)
    elif name == "SB18":
        c = SYSTEM_BATH
        rows = stratified_rows(c["d_B"], c["B"])
        X = make_psi(c["d_B"], c["psi_seed"], k=c["d_S"], dtype="c64")
        ref = oracle.sb_apply(c["d_B"], c["B"], c["seed_HB"], c["seed_B1"], small_hermitian(c["d_S"], c["seed_HS"]),
                              small_hermitian(c["d_S"], c["seed_A"]), c["g"], X, rows=rows)
    else:
        raise KeyError(name)
    _REF[name] = (rows, ref)
    return _REF[name]


def test_c2_full_cache_every_row_and_cached_equals_procedural():
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
    _, ref = oracle_ref("C2")                              # FULL oracle apply: every one of the 65536 rows
    check(phi, ref, 1e-11, "C2 full cache, all rows")
    assert abs(np.linalg.norm(phi) ** 2 - 1.0) < 0.05      # ||H psi||^2 = 1 + O(D^-1/2) for this GUE
    hp = mfh.Hamiltonian(D, B, c["seed"], "c128")
    hp.plan("procedural")
    phi_p = hp.apply(d_psi).cpu().numpy()
    check(phi_p, ref, 1e-11, "C2 operator generated, all rows")
    check(phi, phi_p, 1e-13, "cached vs procedural")        # caching is not an approximation


def test_c2_pair_cache_every_row():
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
    _, ref = oracle_ref("C2")
    check(phi, ref, 1e-11, "C2 pair cache, all rows")


def test_c3_scan_every_row_generated_and_cached():
    """C3 against a FULL oracle scan (all 32768 rows x 16 columns): the tcgen05 generator kernels (configs[2] as
    written: the 496 off-diagonal block pairs generated once for both positions by the two-sided kernel, the 32
    diagonal blocks by the one-sided one) and the same operator from cached complex64 blocks (bulk TMA -> TMEM ->
    tcgen05)."""
    c = CONFIGS["C3"]
    D, B, k = c["D"], c["B"], c["k"]
    Psi = make_psi(D, c["psi_seed"], k=k, dtype="c64")
    lam = lambda_grid(k)
    _, ref = oracle_ref("C3")
    out = {}
    for mode in ("procedural", "full"):
        h = mfh.Hamiltonian(D, B, c["seed"], "c64", kind="diag_plus_gue", seed_h0=c["seed_h0"])
        plan = h.plan(mode, k=k)
        assert plan["chosen"]["mode"] == mode
        if mode == "full":
            assert plan["chosen"]["cache_bytes"] == D * D * 8
        else:
            assert h.get_plan()["two_sided_pairs"] == (D // B) * (D // B - 1) // 2
        Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
        h.destroy()
        for v in range(k):
            check(Phi[:, v], ref[:, v], 1e-4, f"C3 {mode} column {v}")
        out[mode] = Phi
    h0 = oracle.h0_diagonal(D, c["seed_h0"])
    assert rel_l2(out["procedural"][:, 0], h0 * Psi[:, 0].astype(np.complex128)) <= 2e-7   # lambda_0 = 0: phi = h0 (.) psi
    for v in range(1, k):                                   # the two tensor-core kernels against each other, all rows
        assert rel_l2(out["procedural"][:, v], out["full"][:, v]) <= 5e-5, v


@pytest.mark.parametrize("mode", ["procedural", "pairs"])
def test_c3_two_sided_kernels_repeat_bit_identically(mode):
    """Race check of the two-sided tensor-core kernels at full size (compute-sanitizer is closed on this pool, DESIGN.md
    section 10): 100 applies from a periodically poisoned workspace must be bit-identical (the kernels hand tiles, unit
    images, TMEM stages and accumulators between 24 warps through 15 mbarriers and 4 named barriers; the race of round 1
    showed as sporadic wrong rows at full size only) and no guard byte around the library's buffers may change."""
    import torch
    c = CONFIGS["C3"]
    D, B, k = c["D"], c["B"], c["k"]
    Psi = to_dev(make_psi(D, c["psi_seed"], k=k, dtype="c64"))
    lam = lambda_grid(k)
    h = mfh.Hamiltonian(D, B, c["seed"], "c64", kind="diag_plus_gue", seed_h0=c["seed_h0"])
    h.plan(mode, k=k)
    first = h.apply(Psi, lambdas=lam).clone()
    out = torch.empty_like(first)
    for r in range(100):
        if r % 10 == 0:
            h.debug_poison()
        h.apply(Psi, out, lambdas=lam)
        assert torch.equal(out, first), r
    assert h.debug_selfcheck() == 0
    h.destroy()


def test_c3_scan_from_the_pair_cache_every_row():
    """C3's operator from the Hermitian pair cache (4.4 GB instead of 8.6 GB): every stored off-diagonal block is read
    ONCE per apply and serves both positions (two-sided cached kernel, unit-image layout); the diagonal blocks go
    through the one-sided cached kernel."""
    c = CONFIGS["C3"]
    D, B, k = c["D"], c["B"], c["k"]
    Psi = make_psi(D, c["psi_seed"], k=k, dtype="c64")
    lam = lambda_grid(k)
    _, ref = oracle_ref("C3")
    h = mfh.Hamiltonian(D, B, c["seed"], "c64", kind="diag_plus_gue", seed_h0=c["seed_h0"])
    plan = h.plan("pairs", k=k)
    N = D // B
    assert plan["chosen"]["mode"] == "pairs" and plan["chosen"]["cache_bytes"] == N * (N + 1) // 2 * B * B * 8
    assert h.get_plan()["two_sided_stored_pairs"] == N * (N - 1) // 2
    Phi = h.apply(to_dev(Psi), lambdas=lam).cpu().numpy()
    h.destroy()
    for v in range(k):
        check(Phi[:, v], ref[:, v], 1e-4, f"C3 pair cache column {v}")


def test_c3_scan_from_cached_complex128_blocks_stratified_rows():
    """C3's operator cached in double precision (17.2 GB -> FP64 CUDA-core k-vector kernel)."""
    c = CONFIGS["C3"]
    D, B, k = c["D"], c["B"], c["k"]
    lam = lambda_grid(k)
    rows, ref = oracle_ref("C3-c128")
    assert len(rows) >= 8192
    Psi = make_psi(D, c["psi_seed"], k=k, dtype="c128")
    h = mfh.Hamiltonian(D, B, c["seed"], "c128", kind="diag_plus_gue", seed_h0=c["seed_h0"])
    plan = h.plan("full", k=k)
    assert plan["chosen"]["cache_bytes"] == D * D * 16
    d_Psi = to_dev(Psi)
    Phi_t = h.apply(d_Psi, lambdas=lam).clone()
    h.destroy()
    Phi = Phi_t.cpu().numpy()
    for v in range(k):
        check(Phi[rows, v], ref[:, v], 1e-11, f"C3 c128 cached column {v}")
    # every row: the generated complex128 scan (CUDA-core kernel) must agree with the cached one
    hp = mfh.Hamiltonian(D, B, c["seed"], "c128", kind="diag_plus_gue", seed_h0=c["seed_h0"])
    hp.plan("procedural", k=k)
    Phi_p = hp.apply(d_Psi, lambdas=lam).cpu().numpy()
    hp.destroy()
    for v in range(k):
        check(Phi_p[:, v], Phi[:, v], 1e-12 if v else 1e-11, f"C3 c128 generated vs cached column {v}")


def test_c4_procedural_stratified_rows():
    c = CONFIGS["C4"]
    D, B = c["D"], c["B"]
    psi = make_psi(D, c["psi_seed"])
    h = mfh.Hamiltonian(D, B, c["seed"], "c128")
    plan = h.plan("procedural", n_applies_hint=10)
    assert plan["chosen"]["mode"] == "procedural" and plan["dense_bytes"] == D * D * 16
    phi = h.apply(to_dev(psi)).cpu().numpy()
    rows, ref = oracle_ref("C4")
    assert len(rows) >= 8192 and len(set(rows % 128)) == 128 and len(set(rows // B)) == D // B
    check(phi[rows], ref, 1e-11, "C4 procedural")
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
    phi_t = h.apply(d_psi).clone()
    phi = phi_t.cpu().numpy()
    rows, ref = oracle_ref("C5")
    assert len(rows) >= 8192
    check(phi[rows], ref, 1e-11, "C5 partial cache")
    out, K = h.chebyshev(d_psi, c["t"], c["e_min"], c["e_max"], c["tol"])
    assert K == 152 == oracle.chebyshev_n_terms(2.1 * c["t"], c["tol"])
    nrm = float(torch.linalg.vector_norm(out).item())
    assert abs(nrm - 1.0) <= 1e-10                          # BASELINE.json configs[4]
    back, _ = h.chebyshev(out, -c["t"], c["e_min"], c["e_max"], c["tol"])
    assert rel_l2(back.cpu().numpy(), psi) <= 1e-10         # time reversal (Eq. 40 unitarity)
    h.destroy()
    del out, back
    torch.cuda.empty_cache()
    # every row: the partial-cache kernels against the purely generated operator (caching changes nothing)
    hp = mfh.Hamiltonian(D, B, c["seed"], "c128")
    hp.plan("procedural")
    phi_p = hp.apply(d_psi).cpu().numpy()
    hp.destroy()
    check(phi_p[rows], ref, 1e-11, "C5 operator generated")
    check(phi, phi_p, 1e-13, "C5 partial vs procedural, all rows")


def test_c5_pair_cache_stratified_rows_and_every_row_vs_procedural():
    import torch
    c = CONFIGS["C5"]
    D, B = c["D"], c["B"]
    if free_bytes() < 160e9:
        pytest.skip("needs ~150 GB of free HBM")
    psi = make_psi(D, c["psi_seed"])
    d_psi = to_dev(psi)
    h = mfh.Hamiltonian(D, B, c["seed"], "c128")
    plan = h.plan("pairs", n_applies_hint=151, hbm_budget_bytes=int(c["hbm_budget"]))
    assert plan["chosen"]["mode"] == "pairs" and plan["chosen"]["cached_fraction"] == 1.0
    phi = h.apply(d_psi).cpu().numpy()
    h.destroy()
    torch.cuda.empty_cache()
    rows, ref = oracle_ref("C5")
    check(phi[rows], ref, 1e-11, "C5 pair cache")
    hp = mfh.Hamiltonian(D, B, c["seed"], "c128")
    hp.plan("procedural")
    phi_p = hp.apply(d_psi).cpu().numpy()
    hp.destroy()
    check(phi, phi_p, 1e-13, "C5 pairs vs procedural, all rows")


def test_c5_partial_pair_cache_every_row_vs_procedural():
    """A pair cache that does NOT hold the whole operator (the regime beyond C5: D >= 2^18 in complex128): stored
    pairs and generated pairs in one apply."""
    import torch
    c = CONFIGS["C5"]
    D, B = c["D"], c["B"]
    if free_bytes() < 80e9:
        pytest.skip("needs ~75 GB of free HBM")
    psi = make_psi(D, c["psi_seed"])
    d_psi = to_dev(psi)
    h = mfh.Hamiltonian(D, B, c["seed"], "c128")
    plan = h.plan("pairs", n_applies_hint=151, hbm_budget_bytes=int(75e9))
    assert plan["chosen"]["mode"] == "pairs" and 0.3 < plan["chosen"]["cached_fraction"] < 0.7
    phi = h.apply(d_psi).cpu().numpy()
    h.destroy()
    torch.cuda.empty_cache()
    rows, ref = oracle_ref("C5")
    check(phi[rows], ref, 1e-11, "C5 partial pair cache")
    hp = mfh.Hamiltonian(D, B, c["seed"], "c128")
    hp.plan("procedural")
    phi_p = hp.apply(d_psi).cpu().numpy()
    hp.destroy()
    check(phi, phi_p, 1e-13, "C5 partial pairs vs procedural, all rows")


def test_complex64_partial_cache_mid_size_every_row():
    """The partial-cache kernel in complex64 (streaming role: 16-byte unit = two entries) beyond the small shapes of
    the sweep: D = 32768, B = 1024, half the blocks cached, against a full oracle apply and the generated operator."""
    D, B, seed = 32768, 1024, 77
    psi = make_psi(D, 5, dtype="c64")
    ref = oracle.apply(D, B, seed, psi)
    h = mfh.Hamiltonian(D, B, seed, "c64")
    plan = h.plan("partial", n_applies_hint=100, hbm_budget_bytes=int(0.5 * D * D * 8))
    assert plan["chosen"]["mode"] == "partial" and 0.3 < plan["chosen"]["cached_fraction"] < 0.6
    assert h.get_plan()["launches_per_apply"] == 2 and h.get_plan()["stream_sms"] > 0
    d_psi = to_dev(psi)
    phi = h.apply(d_psi).cpu().numpy()
    h.destroy()
    check(phi, ref, 1e-4, "c64 partial cache, all rows")
    hp = mfh.Hamiltonian(D, B, seed, "c64")
    hp.plan("procedural")
    phi_p = hp.apply(d_psi).cpu().numpy()
    hp.destroy()
    check(phi, phi_p, 2e-6, "c64 partial vs generated, all rows")


def test_system_bath_paper_size_stratified_rows_and_c64_vs_c128():
    """The paper's 18-qubit shape: d_S = 4, d_B = 65536, complex64, two cached operators of 32 GiB."""
    import torch
    c = SYSTEM_BATH
    if free_bytes() < 80e9:
        pytest.skip("needs 69 GB of free HBM")
    d_B, d_S, B = c["d_B"], c["d_S"], c["B"]
    H_S, A = small_hermitian(d_S, c["seed_HS"]), small_hermitian(d_S, c["seed_A"])
    X = make_psi(d_B, c["psi_seed"], k=d_S, dtype="c64")
    sb = mfh.SystemBath(d_B, d_S, B, c["seed_HB"], c["seed_B1"], H_S, A, c["g"], dtype="c64")
    plan = sb.plan(c["mode"])
    assert plan["H_B"]["cached_fraction"] == 1.0 and plan["B_1"]["cached_fraction"] == 1.0
    assert plan["flops_per_apply"] == pytest.approx(2.749e11, rel=1e-3)      # 2 * 4 * 65536^2 * 8
    Y = sb.apply(to_dev(X)).cpu().numpy()
    sb.destroy()
    torch.cuda.empty_cache()
    rows, ref = oracle_ref("SB18")
    assert len(rows) >= 8192
    for s in range(d_S):
        check(Y[rows, s], ref[:, s], 1e-4, f"SB18 column {s}")
    # the same two operators from Hermitian pair caches (2 x 17.2 GB instead of 2 x 34.4 GB)
    sbp = mfh.SystemBath(d_B, d_S, B, c["seed_HB"], c["seed_B1"], H_S, A, c["g"], dtype="c64")
    planp = sbp.plan("pairs")
    assert planp["H_B"]["mode"] == "pairs" and planp["H_B"]["cache_bytes"] == (d_B // B) * (d_B // B + 1) // 2 * B * B * 8
    Yp = sbp.apply(to_dev(X)).cpu().numpy()
    sbp.destroy()
    torch.cuda.empty_cache()
    for s in range(d_S):
        check(Yp[rows, s], ref[:, s], 1e-4, f"SB18 pair caches column {s}")
        check(Yp[:, s], Y[:, s], 5e-5, f"SB18 pair caches vs full caches, all rows, column {s}")
    # every row: the same action in complex128 with both operators generated (CUDA-core k-vector kernel)
    sb2 = mfh.SystemBath(d_B, d_S, B, c["seed_HB"], c["seed_B1"], H_S, A, c["g"], dtype="c128")
    sb2.plan("procedural")
    Y2 = sb2.apply(to_dev(X.astype(np.complex128))).cpu().numpy()
    sb2.destroy()
    for s in range(d_S):
        check(Y2[rows, s], ref[:, s], 1e-11, f"SB18 c128 generated column {s}")
        check(Y[:, s], Y2[:, s], 1e-4, f"SB18 c64 cached vs c128 generated, all rows, column {s}")


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


def test_chebyshev_large_argument_R_t_above_1000():
    """a = R t = 1500: about 1600 terms.  The Bessel table must stay accurate there (Miller recurrence; the C++17
    special function breaks down for x > 1000); exact reference by eigh."""
    D, B = 512, 128
    t, e0, e1, tol = 1500.0 / 2.1, -2.1, 2.1, 1e-13
    psi = make_psi(D, 7)
    h = mfh.Hamiltonian(D, B, 21, "c128")
    h.plan("full")
    out, K = h.chebyshev(to_dev(psi), t, e0, e1, tol)
    assert K == oracle.chebyshev_n_terms(2.1 * t, tol) and 1500 < K < 1700
    H = oracle.materialize(D, 21)
    w, U = np.linalg.eigh(H)
    exact = U @ (np.exp(-1j * w * t) * (U.conj().T @ psi))
    got = out.cpu().numpy()
    assert np.all(np.isfinite(got.view(np.float64)))
    assert rel_l2(got, exact) <= 5e-11
    assert abs(np.linalg.norm(got) - 1.0) <= 1e-10
    h.destroy()


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
    rows = lo + stratified_rows(cnt, B, n_min=2048)        # every 128-row tile of the slab, every residue mod 128
    ref = oracle.apply(D, B, c["seed"], psi_np, rows=rows)
    check(got[rows], ref, 1e-11, "C4 row slab of rank 5 of 8")
    assert np.all(got[:lo] == 3.0 - 4.0j) and np.all(got[lo + cnt:] == 3.0 - 4.0j)
    assert rel_l2(got[lo:lo + cnt], full.cpu().numpy()[lo:lo + cnt]) <= 1e-13
    hr.destroy()
