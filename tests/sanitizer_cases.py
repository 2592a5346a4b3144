#!/usr/bin/env python
"""One small case of every kernel of the library, each checked against the CPU oracle AND by the library's own
self-checks (SURVEY.md section 5 "Race detection"; profiles/r02_sanitizer.md):

    python tests/sanitizer_cases.py                      # also run by tests/test_gpu_selfcheck.py under pytest -m gpu
    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py      # where the tool is available
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool initcheck python tests/sanitizer_cases.py

compute-sanitizer is CLOSED on the GPU pool this build runs on (its answer is quoted in profiles/r02_sanitizer.md),
so every apply of every case is wrapped in the substitutes the library offers itself (include/mfh.h, self-check
exports):
  * initcheck  -> the partial-sum workspace, the Chebyshev scratch and the output vector are filled with NaN before
                  the apply: a read of anything this apply did not write makes the result NaN and fails parity;
  * racecheck  -> the apply is repeated three times from the poisoned state and must be bit-identical (a data race
                  between warps or CTAs shows as a run-to-run difference), the result must match the oracle;
  * memcheck   -> every library-owned buffer sits between two 4 KB guard bands; after the applies no guard byte may
                  have changed (out-of-bounds writes), and the caller-owned output has its own guard bands here.
Exits non-zero on any failure.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2606_31598_b200 import binding as mfh  # noqa: E402
from paper_2606_31598_b200.inputs import dense_matrix, lambda_grid, make_psi, small_hermitian  # noqa: E402


def rel(a, b):
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def checked_apply(h, psi, lambdas=None, repeats=3):
    """h.apply under the self-checks of the module docstring; returns phi as numpy."""
    import torch
    n, pad = psi.numel(), 512
    first = None
    for _ in range(repeats):
        buf = torch.full((n + 2 * pad,), float("nan"), dtype=psi.dtype, device="cuda")
        buf[:pad] = 7.0 - 3.0j
        buf[n + pad:] = 7.0 - 3.0j
        phi = buf[pad:pad + n].view(psi.shape)
        h.debug_poison()
        h.apply(psi, phi, lambdas=lambdas)
        torch.cuda.synchronize()
        assert bool(torch.all(buf[:pad] == 7.0 - 3.0j)) and bool(torch.all(buf[n + pad:] == 7.0 - 3.0j)), "write outside phi"
        assert not bool(torch.isnan(torch.view_as_real(phi)).any()), "NaN in phi: something read what this apply did not write"
        if first is None:
            first = phi.clone()
        else:
            assert torch.equal(phi, first), "repeated applies differ bit for bit"
    bad = h.debug_selfcheck()
    assert bad == 0, f"{bad} guard bytes around the library's buffers were overwritten"
    return first.cpu().numpy()


def main(only=None):
    import torch
    assert torch.cuda.is_available()
    dev = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()  # noqa: E731
    done = []

    def case(name, err, tol):
        print(f"sanitizer case {name:44s} rel L2 = {err:.3e}", flush=True)
        assert err <= tol, (name, err)
        done.append(name)

    want = lambda tag: only is None or tag in only  # noqa: E731

    if want("c1"):
        # BASELINE config 1 in the four storage modes: proc_single_kernel, cached_kernel_c128, partial_overlap_kernel,
        # cached_pairs_kernel (+ fill_kernel, reduce_kernel)
        D, B, seed = 4096, 512, 1234
        psi = make_psi(D, 99)
        ref = oracle.apply(D, B, seed, psi)
        for mode, budget in (("procedural", 0), ("full", 0), ("partial", 150_000_000), ("pairs", 0), ("pairs", 90_000_000)):
            h = mfh.Hamiltonian(D, B, seed, "c128")
            p = h.plan(mode, hbm_budget_bytes=budget)
            case(f"C1 c128 {mode} ({p['chosen']['cached_fraction']:.2f} cached)", rel(checked_apply(h, dev(psi)), ref), 1e-11)
            h.destroy()

    if want("c64"):
        # complex64, one vector: proc_single_kernel<float>, cached_kernel_c64, cached_pairs_kernel<float>
        D, B, seed = 2048, 256, 5
        psi = make_psi(D, 3, dtype="c64")
        ref = oracle.apply(D, B, seed, psi)
        for mode, budget in (("procedural", 0), ("full", 0), ("partial", 20_000_000), ("pairs", 0)):
            h = mfh.Hamiltonian(D, B, seed, "c64")
            h.plan(mode, hbm_budget_bytes=budget)
            case(f"c64 k=1 {mode}", rel(checked_apply(h, dev(psi)), ref), 1e-4)
            h.destroy()

    if want("scan"):
        # k = 16 complex64 scan: pairs_tc_kernel<false> (block pairs generated once for both positions) + proc_multi_tc_kernel
        # (diagonal blocks; tcgen05, A generated into TMEM), cached_multi_tc_kernel (bulk TMA), pairs_tc_kernel<true> (pair cache),
        # and a partial k-vector plan (both in one apply)
        D, B, k = 2048, 256, 16
        Psi = make_psi(D, 9, k=k, dtype="c64")
        lam = lambda_grid(k)
        ref = oracle.apply_scan(D, B, 8, 7, lam, Psi)
        for mode, budget in (("procedural", 0), ("full", 0), ("partial", 24_000_000), ("pairs", 0)):
            h = mfh.Hamiltonian(D, B, 8, "c64", kind="diag_plus_gue", seed_h0=7)
            try:
                h.plan(mode, k=k, hbm_budget_bytes=budget)
            except mfh.MfhError as e:
                print(f"sanitizer case c64 k=16 {mode}: not planned ({e})")
                continue
            Phi = checked_apply(h, dev(Psi), lam)
            case(f"c64 k=16 scan {mode}", max(rel(Phi[:, v], ref[:, v]) for v in range(k)), 1e-4)
            h.destroy()

    if want("c128k"):
        # complex128 k-vector kernels: cached_multi_kernel_c128 (k = 16: two threads per row; k = 4), proc_multi_kernel
        D, B = 1024, 256
        for k in (16, 4):
            Psi = make_psi(D, 9, k=k)
            lam = lambda_grid(k)
            ref = oracle.apply_scan(D, B, 8, 7, lam, Psi)
            for mode in ("full", "procedural"):
                h = mfh.Hamiltonian(D, B, 8, "c128", kind="diag_plus_gue", seed_h0=7)
                h.plan(mode, k=k)
                Phi = checked_apply(h, dev(Psi), lam)
                case(f"c128 k={k} {mode}", max(rel(Phi[:, v], ref[:, v]) for v in range(k)), 1e-11)
                h.destroy()

    if want("cheb"):
        # chained drivers: Chebyshev (real and imaginary time, steps), Lanczos; cheb_* and lz_* kernels
        D, B = 1024, 256
        psi = make_psi(D, 99)
        H = oracle.materialize(D, 21)
        h = mfh.Hamiltonian(D, B, 21, "c128")
        h.plan("pairs")
        h.debug_poison()
        out, K = h.chebyshev(dev(psi), 5.0, -2.1, 2.1, 1e-14)
        ref, Kr = oracle.chebyshev_propagate(lambda v: H @ v, psi, 5.0, -2.1, 2.1, 1e-14)
        assert K == Kr
        case("Chebyshev t=5 (pair cache)", rel(out.cpu().numpy(), ref), 1e-11)
        out2, _ = h.chebyshev_steps(dev(psi), 2.5, 2, -2.1, 2.1, 1e-14)
        case("Chebyshev 2 steps of 2.5", rel(out2.cpu().numpy(), ref), 1e-11)
        outi, Ki = h.chebyshev_imag(dev(psi), 3.0, -2.1, 2.1, 1e-13)
        refi, _ = oracle.chebyshev_imag_propagate(lambda v: H @ v, psi, 3.0, -2.1, 2.1, 1e-13)
        case("imaginary-time filter beta=3", float(np.linalg.norm(outi.cpu().numpy() - refi)), 1e-11)
        e0, e1, al, be = h.lanczos_bounds(dev(psi), m=12)
        ro = oracle.lanczos_bounds(lambda v: H @ v, psi, m=12)
        case("Lanczos bounds m=12", max(abs(e0 - ro[0]), abs(e1 - ro[1])), 1e-8)
        assert h.debug_selfcheck() == 0
        h.destroy()

    if want("sb"):
        # system-bath action (mfh_sb_*): two cached operators on d_S columns + the mixing kernel
        d_B, d_S, B, g = 1024, 4, 256, 0.6
        H_S, A = small_hermitian(d_S, 33), small_hermitian(d_S, 34)
        X = make_psi(d_B, 35, k=d_S, dtype="c64")
        sb = mfh.SystemBath(d_B, d_S, B, 31, 32, H_S, A, g, dtype="c64")
        sb.plan("full")
        Y = sb.apply(dev(X)).cpu().numpy()
        ref = oracle.sb_apply(d_B, B, 31, 32, H_S, A, g, X)
        case("system-bath c64 cached d_S=4", max(rel(Y[:, s], ref[:, s]) for s in range(d_S)), 1e-4)
        sb.destroy()

    if want("src"):
        # analytic source (Eq. 9) and externally stored blocks (Eq. 10, retile_kernel for the tiled cache)
        D, B = 1024, 256
        psi = make_psi(D, 4)
        theta = (1.0, 1.3, 0.4, 0.8, 0.61803398875, 0.2)
        h = mfh.Hamiltonian(D, B, 0, "c128", kind="analytic")
        h.set_source_params(theta)
        h.plan("partial", hbm_budget_bytes=12_000_000)
        case("analytic source partial", rel(checked_apply(h, dev(psi)), oracle.analytic_apply(D, theta, psi)), 1e-11)
        h.destroy()
        M = dense_matrix(D, 77)
        k = 4
        Psi = make_psi(D, 6, k=k, dtype="c64")
        h = mfh.Hamiltonian(D, B, 0, "c64", kind="external")
        h.plan("full", k=k)
        for n in range(D // B):
            for m in range(D // B):
                h.set_block(n, m, np.ascontiguousarray(M[n * B:(n + 1) * B, m * B:(m + 1) * B]).astype(np.complex64))
        Phi = checked_apply(h, dev(Psi))
        ref = M.astype(np.complex64).astype(np.complex128) @ Psi.astype(np.complex128)
        case("external blocks c64 k=4 (tiled cache)", max(rel(Phi[:, v], ref[:, v]) for v in range(k)), 1e-4)
        h.destroy()

    torch.cuda.synchronize()
    print(f"sanitizer cases: {len(done)} OK")


if __name__ == "__main__":
    main(set(sys.argv[1:]) or None)
