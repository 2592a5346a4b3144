"""N > 1 path of distributed execution on CPU (world size 2 and 3, gloo, 127.0.0.1): the exchange step of
paper_2606_31598_b200/distributed.py -- all-gather of row slabs ("rows", equal and ragged) and all-reduce
of partial vectors ("pairs") -- driven with the ORACLE's per-rank contributions, must leave the complete
phi = H psi on every rank.  (The per-rank contributions of the CUDA path are checked against the same
oracle contributions in tests/test_gpu_partition.py.)"""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["MFH_ROOT"])
import numpy as np, torch
import torch.distributed as dist
import oracle
from paper_2606_31598_b200.distributed import exchange, slab
from paper_2606_31598_b200.inputs import make_psi
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
D, B, seed = 256, 32, 1234
n_blk = D // B
for k in (1, 4):
    psi = make_psi(D, 99, k=k)
    ref = oracle.apply(D, B, seed, psi)
    for scheme in ("rows", "pairs"):
        part = oracle.apply_partition(D, B, seed, psi, rank, world, scheme)
        lo, hi = slab(n_blk, rank, world) if scheme == "rows" else (0, n_blk)
        if scheme == "rows":                      # rows outside the slab are undefined on the product side
            part = part.copy()
            mask = np.ones(D, dtype=bool); mask[lo * B:hi * B] = False
            part[mask] = 123.0
        phi = torch.from_numpy(part.copy())                # exchange works in place
        out = exchange(phi, scheme, (lo * B, (hi - lo) * B)).numpy()
        err = np.linalg.norm(out - ref) / np.linalg.norm(ref)
        assert err < 1e-13, (scheme, k, err)
        # the real view the library's hook passes: [D][2k] doubles
        phi2 = torch.view_as_real(torch.from_numpy(part.copy()).reshape(D, k)).reshape(D, 2 * k)
        out2 = torch.view_as_complex(exchange(phi2, scheme, (lo * B, (hi - lo) * B)).reshape(D, k, 2)).numpy()
        assert np.linalg.norm(out2.reshape(ref.shape) - ref) / np.linalg.norm(ref) < 1e-13
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_completes_phi_on_every_rank(world):
    port = _free_port()
    procs = []
    for rank in range(world):
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                   WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MFH_ROOT=ROOT, OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for rank, p in enumerate(procs):
        out, _ = p.communicate(timeout=600)
        assert p.returncode == 0 and f"ok {rank}" in out, out


HYBRID_WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["MFH_ROOT"])
import numpy as np, torch
import torch.distributed as dist
import oracle
from paper_2606_31598_b200.distributed import exchange, make_group, my_tasks, slab
from paper_2606_31598_b200.inputs import make_psi
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
p_row, n_tasks = 2, 5                                   # 2 groups of 2 ranks, 5 coupling values -> 3 waves
group, g, C = make_group(p_row)
assert C == world // p_row and g == rank // p_row
gr = dist.get_rank(group)
D, B, seed = 256, 32, 8
n_blk = D // B
lams = np.linspace(0.0, 2.0, n_tasks)
done = {}
for t in my_tasks(n_tasks, g, C):                        # the group's tasks, wave by wave
    psi = make_psi(D, 100 + t)
    for scheme in ("rows", "pairs"):
        part = lams[t] * oracle.apply_partition(D, B, seed, psi, gr, p_row, scheme)
        lo, hi = slab(n_blk, gr, p_row) if scheme == "rows" else (0, n_blk)
        phi = exchange(torch.from_numpy(part.copy()), scheme, (lo * B, (hi - lo) * B), group).numpy()
        ref = lams[t] * oracle.apply(D, B, seed, psi)
        assert np.linalg.norm(phi - ref) <= 1e-13 * max(np.linalg.norm(ref), 1e-300) + 1e-300, (t, scheme)
    done[t] = True
allt = [None] * world
dist.all_gather_object(allt, sorted(done))
assert sorted({t for lst in allt for t in lst}) == list(range(n_tasks))      # every task ran somewhere
assert all(allt[r] == allt[r - r % p_row] for r in range(world))             # the ranks of a group ran the same tasks
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


def test_hybrid_groups_and_task_waves_world_4():
    """Parameter-parallel groups x row-parallel ranks: 4 ranks, row groups of 2, 5 tasks."""
    port = _free_port()
    world = 4
    procs = []
    for rank in range(world):
        env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                   WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MFH_ROOT=ROOT, OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, "-c", HYBRID_WORKER], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.STDOUT, text=True))
    for rank, p in enumerate(procs):
        out, _ = p.communicate(timeout=600)
        assert p.returncode == 0 and f"ok {rank}" in out, out
