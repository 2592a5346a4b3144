"""GPU parity of distributed execution (NEXT-4; mfh_set_partition).

One GPU is enough: the ranks of a job never wait on one another inside an apply (every rank reads the full
psi, the exchange follows), so rank r of W is run as its own handle, one after the other, and each
contribution is compared element by element with the oracle's contribution of the same rank
(oracle/partition.py states the ownership rule independently)."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200.inputs import lambda_grid, make_psi

pytestmark = pytest.mark.gpu

TOL = {"c128": 1e-11, "c64": 1e-4}
SENTINEL = 7.25 - 3.5j


def to_dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def rank_apply(D, B, seed, psi, dtype, mode, rank, world, scheme, k=1, budget=0, lambdas=None, **kw):
    """Contribution of one rank: phi prefilled with a sentinel so that untouched rows show."""
    import torch
    h = mfh.Hamiltonian(D, B, seed, dtype, **kw)
    h.set_partition(rank, world, scheme)
    h.plan(mode, k=k, hbm_budget_bytes=budget)
    plan = h.get_plan()
    x = to_dev(psi)
    phi = torch.full_like(x, SENTINEL)
    h.apply(x, phi, lambdas)
    out = phi.cpu().numpy().astype(np.complex128)
    lo, cnt = h.partition_rows()
    h.destroy()
    return out, plan, (lo, cnt)


def scaled_err(a, b, scale):
    return float(np.linalg.norm(a - b) / scale)


@pytest.mark.parametrize("scheme", ["rows", "pairs"])
@pytest.mark.parametrize("mode", ["procedural", "partial", "full", "pairs"])
@pytest.mark.parametrize("dtype", ["c128", "c64"])
@pytest.mark.parametrize("world", [2, 3])
def test_each_rank_matches_the_oracle_contribution(scheme, mode, dtype, world):
    D, B, seed = 2048, 256, 1234                                   # 8 x 8 blocks, ragged at world 3
    psi = make_psi(D, 99, dtype=dtype)
    full = oracle.apply(D, B, seed, psi)
    scale = np.linalg.norm(full)
    budget = int(0.45 * D * D * (16 if dtype == "c128" else 8) / world) if mode == "partial" else 0
    total = np.zeros(D, dtype=np.complex128)
    for r in range(world):
        got, plan, (lo, cnt) = rank_apply(D, B, seed, psi, dtype, mode, r, world, scheme, budget=budget)
        ref = oracle.apply_partition(D, B, seed, psi, r, world, scheme)
        assert plan["partition"]["rank"] == r and plan["partition"]["world"] == world
        assert plan["partition"]["owned_blocks"] == int(oracle.owned_blocks(D // B, r, world, scheme).sum())
        if scheme == "rows":
            assert (lo, cnt) == (B * (8 * r // world), B * (8 * (r + 1) // world) - B * (8 * r // world))
            outside = np.ones(D, dtype=bool)
            outside[lo:lo + cnt] = False
            assert np.all(got[outside] == SENTINEL)                # foreign rows untouched
            got = np.where(outside, 0.0, got)
        else:
            assert (lo, cnt) == (0, D)
        assert scaled_err(got, ref, scale) <= TOL[dtype], (r, plan)
        total += got
    assert scaled_err(total, full, scale) <= TOL[dtype]


@pytest.mark.parametrize("scheme", ["rows", "pairs"])
def test_coupling_scan_k_vectors_partitioned(scheme):
    """H0 + lambda_v V with k = 16 (complex64, tensor-core kernels): the H0 term appears exactly once."""
    D, B, k, world = 2048, 256, 16, 2
    Psi = make_psi(D, 9, k=k, dtype="c64")
    lam = lambda_grid(k)
    full = oracle.apply_scan(D, B, 8, 7, lam, Psi)
    for mode in ("procedural", "full"):
        total = np.zeros((D, k), dtype=np.complex128)
        for r in range(world):
            got, plan, (lo, cnt) = rank_apply(D, B, 8, Psi, "c64", mode, r, world, scheme, k=k, lambdas=lam,
                                              kind="diag_plus_gue", seed_h0=7)
            if scheme == "rows":
                outside = np.ones(D, dtype=bool)
                outside[lo:lo + cnt] = False
                got[outside] = 0.0
            total += got
        for v in range(k):
            err = np.linalg.norm(total[:, v] - full[:, v]) / np.linalg.norm(full[:, v])
            assert err <= 1e-4, (mode, v, err)


def test_world_8_pairs_procedural_c128_sum_and_balance():
    """C1's operator over 8 ranks: contributions add up to the full apply; the generation work is even."""
    D, B, seed, world = 4096, 256, 1234, 8                          # 16 x 16 blocks: 136 pairs, 17 per rank
    psi = make_psi(D, 99)
    full = oracle.apply(D, B, seed, psi)
    total = np.zeros(D, dtype=np.complex128)
    items = []
    for r in range(world):
        got, plan, _ = rank_apply(D, B, seed, psi, "c128", "procedural", r, world, "pairs")
        total += got
        items.append(plan["proc_items"])
    assert np.linalg.norm(total - full) <= 1e-11 * np.linalg.norm(full)
    assert max(items) - min(items) <= max(items) // 8 + 1


def test_invalid_partition_arguments_and_replan():
    h = mfh.Hamiltonian(1024, 128, 1, "c128")
    for args in [(2, 2, "rows"), (-1, 2, "pairs"), (0, 0, "rows"), (0, 2, "none")]:
        with pytest.raises(mfh.MfhError) as e:
            h.set_partition(*args)
        assert e.value.code == mfh.MFH_ERR_INVALID_ARG
    h.plan("procedural")
    h.set_partition(1, 2, "rows")                                   # drops the plan
    with pytest.raises(mfh.MfhError) as e:
        h.apply(to_dev(make_psi(1024, 1)))
    assert e.value.code == mfh.MFH_ERR_BAD_STATE
    h.plan("procedural")
    assert h.partition_rows() == (512, 512)
    h.destroy()


def test_chained_drivers_call_the_exchange_hook():
    """mfh_chebyshev / mfh_lanczos_bounds on a handle with a registered hook: one call per apply, on the
    library-owned vector, and the result is unchanged by an identity exchange.  A partitioned handle
    without a hook refuses to chain."""
    import torch
    from paper_2606_31598_b200.distributed import install_exchange_hook
    D, B = 1024, 128
    psi = to_dev(make_psi(D, 3))
    h = mfh.Hamiltonian(D, B, 21, "c128")
    h.plan("procedural")
    ref, K = h.chebyshev(psi, 3.0, -2.1, 2.1, 1e-12)
    seen = []

    def probe(flat, scheme, rows, group):                            # identity exchange that records its input
        seen.append((tuple(flat.shape), float(torch.linalg.vector_norm(flat))))
        return flat

    import paper_2606_31598_b200.distributed as dmod
    orig = dmod.exchange
    dmod.exchange = probe
    try:
        install_exchange_hook(h, "pairs", (0, D))
        out, K2 = h.chebyshev(psi, 3.0, -2.1, 2.1, 1e-12)
        torch.cuda.synchronize()
    finally:
        dmod.exchange = orig
    assert K2 == K and h._exchange_state["calls"] == K - 1 and "error" not in h._exchange_state
    assert all(s[0] == (D, 2) and s[1] > 0 for s in seen)
    assert torch.equal(out, ref)
    h.destroy()

    h2 = mfh.Hamiltonian(D, B, 21, "c128")
    h2.set_partition(0, 2, "pairs")
    h2.plan("procedural")
    with pytest.raises(mfh.MfhError) as e:
        h2.chebyshev(psi, 1.0, -2.1, 2.1, 1e-10)
    assert e.value.code == mfh.MFH_ERR_BAD_STATE
    h2.destroy()


def test_bench_partition_mode_runs_on_one_gpu():
    """bench.py --partition: the sharded-job arm (DistributedHamiltonian + NCCL exchange) with a single-rank
    group; the line must carry the contract keys and the C1 throughput of the plain arm's order."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--workload", "C1", "--partition", "pairs",
                        "--steps", "5", "--warmup", "3"], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    line = json.loads(r.stdout.strip().splitlines()[-1])
    assert line["scaling"] == "strong" and line["n_gpus"] == 1 and line["config"]["partition"]["scheme"] == "pairs"
    assert line["value"] > 1e10 and line["gpu_launches"] > 0


_NCCL_WORLD1 = r"""
import os, socket, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_2606_31598_b200 import binding as mfh
from paper_2606_31598_b200 import distributed as dmod
from paper_2606_31598_b200.inputs import make_psi
with socket.socket() as sk:
    sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]
torch.cuda.set_device(0)
dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1, device_id=torch.device("cuda", 0))
calls = {"all_reduce": 0, "all_gather_into_tensor": 0}
for name in calls:                                    # count the collectives that reach the backend
    orig = getattr(dist, name)
    def wrap(*a, _o=orig, _n=name, **k):
        calls[_n] += 1
        return _o(*a, **k)
    setattr(dist, name, wrap)
D, B = 2048, 256
for dtype, k in (("c128", 1), ("c64", 4)):
    psi = torch.from_numpy(make_psi(D, 99, k=k, dtype=dtype)).cuda()
    h = mfh.Hamiltonian(D, B, 21, dtype); h.plan("procedural", k=k)
    ref = h.apply(psi).clone()
    ref_c = h.chebyshev(psi, 3.0, -2.1, 2.1, 1e-12)[0].clone() if k == 1 else None
    h.destroy()
    for scheme in ("pairs", "rows"):
        before = dict(calls)
        dh = dmod.DistributedHamiltonian(D, B, 21, dtype, scheme=scheme)
        dh.plan(mode="procedural", k=k)
        phi = dh.apply(psi)                            # apply + NCCL exchange (in place on the complex tensor)
        torch.cuda.synchronize()
        assert torch.equal(phi, ref), (dtype, scheme)
        key = "all_reduce" if scheme == "pairs" else "all_gather_into_tensor"
        assert calls[key] == before[key] + 1, (calls, before)
        if k == 1:
            out, K = dh.chebyshev(psi, 3.0, -2.1, 2.1, 1e-12)   # the library's driver calls the hook after every apply
            torch.cuda.synchronize()
            st = dh.h._exchange_state
            assert "error" not in st and st["calls"] == K - 1, st
            assert calls[key] == before[key] + 1 + (K - 1)
            assert torch.equal(out, ref_c), (dtype, scheme)
        dh.destroy()
dist.destroy_process_group()
print("NCCL-WORLD1-OK", calls)
"""


def test_exchange_and_chained_hook_on_the_nccl_backend_world_1():
    """distributed.exchange and the mfh_chebyshev exchange hook on the real backend: a single-rank NCCL group issues
    the same collectives as a multi-GPU job (all_reduce on the real view of the complex vector, in-place
    all_gather_into_tensor), in stream order with the library's kernels.  No N > 1 run exists (one GPU per call)."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-c", _NCCL_WORLD1, root], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "NCCL-WORLD1-OK" in r.stdout, (r.stdout[-1500:], r.stderr[-3000:])
