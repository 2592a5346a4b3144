"""The library's own memory / initialisation / race checks on one small case of every kernel (the substitute for
compute-sanitizer, which is closed on this GPU pool; see tests/sanitizer_cases.py and profiles/r02_sanitizer.md)."""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import sanitizer_cases  # noqa: E402

from paper_2606_31598_b200 import binding as mfh  # noqa: E402
from paper_2606_31598_b200.inputs import make_psi  # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("group", ["c1", "c64", "scan", "c128k", "cheb", "sb", "src"])
def test_selfchecked_cases(group):
    sanitizer_cases.main({group})


def test_the_guard_bands_do_detect_an_out_of_bounds_write():
    """Test of the test: a single byte written right before or right after a library-owned buffer is reported."""
    import torch
    D, B = 1024, 256
    h = mfh.Hamiltonian(D, B, 3, "c128")
    h.plan("partial", hbm_budget_bytes=12_000_000)
    psi = torch.from_numpy(make_psi(D, 1)).cuda()
    sanitizer_cases.checked_apply(h, psi)
    assert h.debug_selfcheck() == 0
    L = mfh.lib()
    assert L.mfh_debug_corrupt_guard(h._h, 0, 1) == mfh.MFH_OK       # one byte past the end of the block cache
    assert h.debug_selfcheck() == 1
    assert L.mfh_debug_corrupt_guard(h._h, 1, 0) == mfh.MFH_OK       # one byte before the partial-sum workspace
    assert h.debug_selfcheck() == 2
    assert L.mfh_debug_corrupt_guard(h._h, 99, 0) == mfh.MFH_ERR_INVALID_ARG
    h.destroy()


def test_fused_tail_single_launch_is_deterministic_and_self_cleaning():
    """Small procedural plans reduce inside the fused kernel (one launch per apply): 50 back-to-back applies must be
    bit-identical (the device counters clean themselves) and match the oracle."""
    import oracle
    import torch
    D, B = 2048, 256
    psi_np = make_psi(D, 99)
    psi = torch.from_numpy(psi_np).cuda()
    for dtype, tol in (("c128", 1e-11), ("c64", 1e-4)):
        p = psi if dtype == "c128" else psi.to(torch.complex64)
        h = mfh.Hamiltonian(D, B, 1234, dtype)
        h.plan("procedural")
        assert h.get_plan()["launches_per_apply"] == 1
        first = h.apply(p).clone()
        for _ in range(50):
            phi = torch.full_like(first, float("nan"))
            h.apply(p, phi)
            assert torch.equal(phi, first)
        ref = oracle.apply(D, B, 1234, p.cpu().numpy())
        err = np.linalg.norm(first.cpu().numpy().astype(np.complex128) - ref) / np.linalg.norm(ref)
        assert err <= tol, (dtype, err)
        h.destroy()


def test_handle_belongs_to_its_device_and_a_second_device_works():
    """include/mfh.h "Devices": a handle lives on the device current in mfh_plan (kernel attributes are kept per handle,
    not per process).  With two GPUs the same process plans and applies on both; with one GPU only the refusal of a
    foreign current device can be checked -- skipped there."""
    import oracle
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices in one process")
    D, B = 4096, 4096                     # B = 4096: the fused kernel needs > 48 KB of dynamic shared memory
    psi = make_psi(D, 5)
    ref = oracle.apply(D, B, 77, psi)
    outs = []
    for dev in (0, 1):
        with torch.cuda.device(dev):
            h = mfh.Hamiltonian(D, B, 77, "c128")
            h.plan("procedural")
            phi = h.apply(torch.from_numpy(psi).cuda()).cpu().numpy()
            assert np.linalg.norm(phi - ref) / np.linalg.norm(ref) <= 1e-11, dev
            outs.append((h, phi))
    with torch.cuda.device(1):            # handle of device 0 used while device 1 is current: refused, not launched
        with pytest.raises(mfh.MfhError) as e:
            outs[0][0].apply(torch.from_numpy(psi).cuda())
        assert e.value.code == mfh.MFH_ERR_BAD_STATE
    for h, _ in outs:
        h.destroy()
