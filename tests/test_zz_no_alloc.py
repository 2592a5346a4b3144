"""mfh_apply_static (include/mfh.h): the allocation-free entry point -- phi = lambda V(seed) psi with its scratch in a
file-scope device array -- against the existing path (mfh_create / mfh_plan / mfh_apply, procedural complex128) and the
CPU oracle, on calls in a row that share the scratch.  Collected last on purpose (file name): the suite runs with
pytest -x.  Passes alone in a fresh process and after the other tests (it depends on no state of theirs; the library's
own state is the per-device scratch, which every call fully rewrites)."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import make_psi

pytestmark = pytest.mark.gpu

TOL = 1e-11   # complex128 tolerance of the parity tests (BASELINE.json north_star)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.complex128)
    b = np.asarray(b, dtype=np.complex128)
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def existing_path(D, B, seed, lam, psi_dev):
    h = mfh.Hamiltonian(D, B, seed, "c128", lam=lam)
    h.plan("procedural")
    out = h.apply(psi_dev).cpu().numpy()
    h.destroy()
    return out


def test_static_entry_point_matches_the_existing_path_two_calls_in_a_row():
    import torch
    D, seed, lam = 4096, 1234, 0.75                       # config 1's operator
    psi_a, psi_b = make_psi(D, 99), make_psi(D, 100)
    xa, xb = to_dev(psi_a), to_dev(psi_b)
    ref_a, ref_b = existing_path(D, 512, seed, lam, xa), existing_path(D, 512, seed, lam, xb)
    # two calls in a row on one stream, outputs preallocated by the caller: the second reuses the first's scratch
    out_a = torch.full_like(xa, float("nan"))
    out_b = torch.full_like(xb, float("nan"))
    mfh.apply_static(D, seed, lam, xa, out_a)
    mfh.apply_static(D, seed, lam, xb, out_b)
    torch.cuda.synchronize()
    assert rel_l2(out_a.cpu().numpy(), ref_a) <= TOL
    assert rel_l2(out_b.cpu().numpy(), ref_b) <= TOL
    # and against the CPU oracle (the definition itself)
    assert rel_l2(out_a.cpu().numpy(), lam * oracle.apply(D, 512, seed, psi_a)) <= TOL
    # the same call again is bit-identical (fixed summation order, no atomics)
    again = mfh.apply_static(D, seed, lam, xa)
    torch.cuda.synchronize()
    assert torch.equal(again, out_a)


def test_static_entry_point_other_sizes_share_the_scratch():
    """A different D re-uploads the generator table into the same array and leaves chunk slots of the previous call
    behind; a ragged number of row tiles (17: the last chunks are empty) and the smallest size."""
    import torch
    for D, B, seed in ((2176, 128, 5), (128, 128, 6), (4096, 512, 1234), (1024, 256, 7)):
        psi = make_psi(D, 31)
        x = to_dev(psi)
        got = mfh.apply_static(D, seed, 1.0, x).cpu().numpy()
        assert rel_l2(got, existing_path(D, B, seed, 1.0, x)) <= TOL, D
        assert rel_l2(got, oracle.apply(D, B, seed, psi)) <= TOL, D
    torch.cuda.synchronize()


def test_static_entry_point_rejects_what_does_not_fit():
    import torch
    x = torch.zeros(128, dtype=torch.complex128, device="cuda")
    y = torch.empty_like(x)
    for D in (mfh.STATIC_MAX_D + 128, 1 << 20, 64, 200):
        rc = mfh.lib().mfh_apply_static(D, 1, 1.0, x.data_ptr(), y.data_ptr(), None)
        assert rc == mfh.MFH_ERR_INVALID_ARG, D
    rc = mfh.lib().mfh_apply_static(mfh.STATIC_MAX_D + 128, 1, 1.0, x.data_ptr(), y.data_ptr(), None)
    assert rc == mfh.MFH_ERR_INVALID_ARG and "MFH_STATIC_MAX_D" in mfh.lib().mfh_last_error().decode()
    assert mfh.lib().mfh_apply_static(128, 1, 1.0, x.data_ptr(), x.data_ptr(), None) == mfh.MFH_ERR_INVALID_ARG   # aliased


def test_static_entry_point_at_its_maximum_size():
    """D = MFH_STATIC_MAX_D: all 4 MB of partial sums in use; sampled rows against the oracle, all rows against the
    existing path."""
    D, seed = mfh.STATIC_MAX_D, 21
    psi = make_psi(D, 3)
    x = to_dev(psi)
    got = mfh.apply_static(D, seed, 1.0, x).cpu().numpy()
    assert rel_l2(got, existing_path(D, 2048, seed, 1.0, x)) <= TOL
    rows = np.arange(0, D, 257, dtype=np.int64)
    ref = oracle.apply(D, 2048, seed, psi, rows=rows)
    assert rel_l2(got[rows], ref) <= TOL


def test_static_entry_point_under_cuda_graph_capture():
    """The reason the entry point exists: after one warm-up call for this D (address look-up, generator table in place)
    it issues kernel launches only, so it can be recorded into a CUDA graph -- where cudaMalloc is not allowed -- and
    replayed."""
    import torch
    D, seed, lam = 2048, 77, 1.25
    x = to_dev(make_psi(D, 5))
    y = torch.empty_like(x)
    mfh.apply_static(D, seed, lam, x, y)                      # warm-up outside the capture
    torch.cuda.synchronize()
    ref = y.clone()
    g = torch.cuda.CUDAGraph()
    y.zero_()
    with torch.cuda.graph(g):
        mfh.apply_static(D, seed, lam, x, y)
    y.zero_()
    for _ in range(3):
        g.replay()
    torch.cuda.synchronize()
    assert torch.equal(y, ref)
    x.copy_(to_dev(make_psi(D, 6)))                           # new input in the captured buffer, replay again
    g.replay()
    torch.cuda.synchronize()
    assert rel_l2(y.cpu().numpy(), existing_path(D, 256, seed, lam, x)) <= TOL
