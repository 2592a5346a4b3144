"""CUDA-graph capture of the hot path: mfh_apply and the chained Chebyshev driver enqueue only kernels and
memsets on the caller's stream (no allocation, no host synchronisation after the first call), so a
launch-bound loop at small D can be captured once and replayed."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import make_psi

pytestmark = pytest.mark.gpu


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("mode", ["procedural", "pairs", "partial"])
def test_apply_replayed_from_a_cuda_graph(mode):
    import torch
    D, B, seed = 4096, 512, 1234                                  # configs[0]
    h = mfh.Hamiltonian(D, B, seed, "c128")
    h.plan(mode, hbm_budget_bytes=int(0.5 * D * D * 16) if mode == "partial" else 0)
    psi = to_dev(make_psi(D, 99))
    phi = torch.empty_like(psi)
    h.apply(psi, phi)                                             # warm-up outside the capture
    eager = phi.clone()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        phi.zero_()
        with torch.cuda.graph(g, stream=s):
            h.apply(psi, phi)
    phi.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(phi, eager)                                # deterministic: bit-identical
    ref = oracle.apply(D, B, seed, make_psi(D, 99))
    assert np.linalg.norm(phi.cpu().numpy() - ref) <= 1e-11 * np.linalg.norm(ref)
    # new input, same graph: the captured launches read the same device pointers
    psi.copy_(to_dev(make_psi(D, 7)))
    g.replay()
    torch.cuda.synchronize()
    ref = oracle.apply(D, B, seed, make_psi(D, 7))
    assert np.linalg.norm(phi.cpu().numpy() - ref) <= 1e-11 * np.linalg.norm(ref)
    h.destroy()


def test_chebyshev_propagation_replayed_from_a_cuda_graph():
    import torch
    D, B, seed = 2048, 256, 21
    h = mfh.Hamiltonian(D, B, seed, "c128")
    h.plan("procedural")
    psi = to_dev(make_psi(D, 3))
    out = torch.empty_like(psi)
    _, K = h.chebyshev(psi, 5.0, -2.1, 2.1, 1e-13, out=out)       # first call allocates the scratch vectors
    eager = out.clone()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            h.chebyshev(psi, 5.0, -2.1, 2.1, 1e-13, out=out)
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out, eager) and K > 10
    h.destroy()
