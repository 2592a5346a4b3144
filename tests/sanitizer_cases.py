#!/usr/bin/env python
"""One small case of every kernel of the library, each checked against the CPU oracle -- the program that
compute-sanitizer runs (SURVEY.md section 5 "Race detection"; profiles/r02_sanitizer.md has the command lines):

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool initcheck python tests/sanitizer_cases.py

Not collected by pytest (no test_ prefix): the same paths are covered, at more shapes, by the -m gpu tests; this
script keeps the launch count low enough for the sanitizer's 10-100x slow-down.  Exits non-zero on a parity failure.
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
            case(f"C1 c128 {mode} ({p['chosen']['cached_fraction']:.2f} cached)", rel(h.apply(dev(psi)).cpu().numpy(), ref), 1e-11)
            h.destroy()

    if want("c64"):
        # complex64, one vector: proc_single_kernel<float>, cached_kernel_c64, cached_pairs_kernel<float>
        D, B, seed = 2048, 256, 5
        psi = make_psi(D, 3, dtype="c64")
        ref = oracle.apply(D, B, seed, psi)
        for mode, budget in (("procedural", 0), ("full", 0), ("partial", 20_000_000), ("pairs", 0)):
            h = mfh.Hamiltonian(D, B, seed, "c64")
            h.plan(mode, hbm_budget_bytes=budget)
            case(f"c64 k=1 {mode}", rel(h.apply(dev(psi)).cpu().numpy(), ref), 1e-4)
            h.destroy()

    if want("scan"):
        # k = 16 complex64 scan: proc_multi_tc_kernel (tcgen05, A generated into TMEM), cached_multi_tc_kernel (bulk TMA),
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
            Phi = h.apply(dev(Psi), lambdas=lam).cpu().numpy()
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
                Phi = h.apply(dev(Psi), lambdas=lam).cpu().numpy()
                case(f"c128 k={k} {mode}", max(rel(Phi[:, v], ref[:, v]) for v in range(k)), 1e-11)
                h.destroy()

    if want("cheb"):
        # chained drivers: Chebyshev (real and imaginary time, steps), Lanczos; cheb_* and lz_* kernels
        D, B = 1024, 256
        psi = make_psi(D, 99)
        H = oracle.materialize(D, 21)
        h = mfh.Hamiltonian(D, B, 21, "c128")
        h.plan("pairs")
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
        case("analytic source partial", rel(h.apply(dev(psi)).cpu().numpy(), oracle.analytic_apply(D, theta, psi)), 1e-11)
        h.destroy()
        M = dense_matrix(D, 77)
        k = 4
        Psi = make_psi(D, 6, k=k, dtype="c64")
        h = mfh.Hamiltonian(D, B, 0, "c64", kind="external")
        h.plan("full", k=k)
        for n in range(D // B):
            for m in range(D // B):
                h.set_block(n, m, np.ascontiguousarray(M[n * B:(n + 1) * B, m * B:(m + 1) * B]).astype(np.complex64))
        Phi = h.apply(dev(Psi)).cpu().numpy()
        ref = M.astype(np.complex64).astype(np.complex128) @ Psi.astype(np.complex128)
        case("external blocks c64 k=4 (tiled cache)", max(rel(Phi[:, v], ref[:, v]) for v in range(k)), 1e-4)
        h.destroy()

    torch.cuda.synchronize()
    print(f"sanitizer cases: {len(done)} OK")


if __name__ == "__main__":
    main(set(sys.argv[1:]) or None)
