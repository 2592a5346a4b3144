"""Distributed phi = H psi over several B200s: one process and one handle per GPU (NEXT-4).

PAPER.md P:185-191: GPU j accumulates phi^[n] = sum_m H^[n,m] psi^[m] for the
block rows (here: block positions) it owns from the FULL psi; "the local outputs can then be gathered";
"the communication volume ... is linear in D, while the dense arithmetic is quadratic in D".

All arithmetic of the apply runs in the library's kernels (``mfh_set_partition`` + ``mfh_apply``); this
module adds the one exchange step per apply, on NCCL through ``torch.distributed`` (NVSwitch: 2-4 MB per
apply, tens of microseconds against 10-100 ms of local work, so a plain collective is the right tool and
no fused kernel is built):

  scheme "rows"   all-gather IN PLACE: rank r wrote rows [lo_r, hi_r) of phi; equal slabs use
                  ``all_gather_into_tensor`` with the local slab as the input view of the output buffer.
  scheme "pairs"  all-reduce (sum) of the full-length partial phi.  Keeps the Hermitian reuse across
                  ranks: a block pair is generated (or stored) once in the whole job, so 2 GPUs halve the
                  generation work, whereas "rows" generates the off-slab blocks one-sided
                  (3/4 of the single-GPU generations per rank at world 2 instead of 1/2).

``exchange`` is device-agnostic (the world-size-2 gloo test drives it with oracle contributions on CPU);
``DistributedHamiltonian`` needs CUDA.  The chained drivers (Chebyshev, Lanczos) stay inside the library:
``install_exchange_hook`` registers the exchange as the handle's hook (``mfh_set_exchange``), which the
library calls after every apply of the chain on the library-owned vector (seen here through the CUDA
array interface, no copy).
"""
from __future__ import annotations


def slab(n_blk: int, rank: int, world: int):
    """Block rows [lo, hi) of rank `rank` under the "rows" scheme (contiguous, sizes differ by at most 1)."""
    return n_blk * rank // world, n_blk * (rank + 1) // world


def exchange(phi, scheme: str, rows, group=None):
    """The exchange step.  phi: full-length tensor [D] or [D,k] holding this rank's contribution
    ("rows": valid on rows[0]:rows[0]+rows[1] only).  On return every rank holds the complete phi."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)   # world 1 issues the same collectives (a single-rank NCCL group exercises the path)
    if scheme == "pairs":
        view = torch.view_as_real(phi) if phi.is_complex() else phi
        dist.all_reduce(view, op=dist.ReduceOp.SUM, group=group)
        return phi
    if scheme != "rows":
        raise ValueError(f"unknown scheme {scheme!r}")
    lo, cnt = rows
    D = phi.shape[0]
    if D % world == 0 and cnt == D // world and lo == dist.get_rank(group) * cnt:
        dist.all_gather_into_tensor(phi, phi[lo:lo + cnt].clone() if phi.device.type == "cpu" else phi[lo:lo + cnt],
                                    group=group)
        return phi
    # ragged slabs: gather (lo, cnt) then the segments
    meta = [None] * world
    dist.all_gather_object(meta, (int(lo), int(cnt)), group=group)
    for r, (l, c) in enumerate(meta):
        if c:
            dist.broadcast(phi[l:l + c], src=dist.get_global_rank(group, r) if group is not None else r, group=group)
    return phi


def row_groups(world: int, p_row: int):
    """GPU groups of a hybrid plan: consecutive ranks form a row group of size p_row,
    e.g. world 8, p_row 2 -> [[0, 1], [2, 3], [4, 5], [6, 7]] (the grouping the paper's run prints)."""
    if p_row < 1 or world % p_row:
        raise ValueError(f"row-group size {p_row} does not divide {world} GPUs")
    return [list(range(g * p_row, (g + 1) * p_row)) for g in range(world // p_row)]


def task_waves(n_tasks: int, n_groups: int):
    """Independent tasks (coupling values, ...) dealt to the groups wave by wave: wave w holds the tasks
    w C .. w C + C - 1, task t runs on group t mod C; len(result) = W(p) = ceil(N_task / C) (Eq. 19)."""
    return [[(t % n_groups, t) for t in range(w * n_groups, min((w + 1) * n_groups, n_tasks))]
            for w in range((n_tasks + n_groups - 1) // n_groups)]


def make_group(p_row: int):
    """Create the process groups of a hybrid plan (collective: every rank calls it) and return
    (this rank's group, its group index, number of groups).  p_row = 1: parameter-parallel, no exchange;
    p_row = world: row-parallel."""
    import torch.distributed as dist
    world, rank = dist.get_world_size(), dist.get_rank()
    mine = None
    groups = row_groups(world, p_row)
    for g, ranks in enumerate(groups):
        pg = dist.new_group(ranks)            # every rank must take part in every new_group call
        if rank in ranks:
            mine = (pg, g)
    return mine[0], mine[1], len(groups)


def my_tasks(n_tasks: int, group_index: int, n_groups: int):
    """The tasks of one group, in wave order."""
    return [t for wave in task_waves(n_tasks, n_groups) for (g, t) in wave if g == group_index]


class _DevicePtr:
    """A library-owned device vector seen through the CUDA array interface (no copy, no ownership)."""

    def __init__(self, ptr: int, n_real: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (n_real,), "typestr": typestr, "data": (ptr, False), "version": 2}


def install_exchange_hook(h, scheme: str, rows, k: int = 1, group=None):
    """Register the exchange of `scheme` as the handle's hook (mfh_set_exchange): the chained drivers
    (mfh_chebyshev, mfh_lanczos_bounds) then call it after every apply.  Returns the ctypes callback
    (also kept alive on the handle object)."""
    import ctypes
    import torch
    from .binding import lib, _check
    real = "<f8" if h.dtype == "c128" else "<f4"
    rsz = 8 if h.dtype == "c128" else 4
    D = h.D
    state = {"calls": 0}

    def _hook(user, phi_dev, nbytes, stream):
        try:
            flat = torch.as_tensor(_DevicePtr(int(phi_dev), int(nbytes) // rsz, real), device="cuda")
            exchange(flat.view(D, 2 * k), scheme, rows, group)     # reals: [D][2k], rows along dim 0
            state["calls"] += 1
            return 0
        except Exception as exc:  # the C side turns a non-zero return into MFH_ERR_CUDA
            state["error"] = exc
            return 1

    FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p)
    cb = FN(_hook)
    lib().mfh_set_exchange.argtypes = [ctypes.c_void_p, FN, ctypes.c_void_p]
    _check(lib().mfh_set_exchange(h._h, cb, None))
    h._exchange_cb, h._exchange_state = cb, state
    return cb


class DistributedHamiltonian:
    """One seeded Hamiltonian spread over the ranks of a process group."""

    def __init__(self, D, B=0, seed=0, dtype="c128", kind="gue", lam=1.0, seed_h0=0, scheme="pairs", group=None):
        import torch.distributed as dist
        from .binding import Hamiltonian
        self.group, self.scheme = group, scheme
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.h = Hamiltonian(D, B, seed, dtype, kind, lam, seed_h0)
        self.h.set_partition(self.rank, self.world, scheme if self.world > 1 else "none")
        self.D = D

    def plan(self, **kw):
        """mfh_plan on every rank.  Block ownership is defined in block indices, so the ranks must agree on B: the
        library refuses B = 0 on a partitioned handle, and the planned (B, n_blk, k) of all ranks are compared here
        (a mismatch would give a silently wrong phi: blocks missing or counted twice)."""
        import torch.distributed as dist
        rec = self.h.plan(**kw)
        self.rows = self.h.partition_rows()
        k = kw.get("k", 1)
        info = self.h.get_plan()
        mine = (int(info["B"]), int(info["n_blk"]), int(info["k"]))
        every = [None] * self.world
        dist.all_gather_object(every, mine, group=self.group)
        if any(tuple(x) != mine for x in every):
            raise RuntimeError(f"ranks planned different block structures (B, n_blk, k): {every}")
        install_exchange_hook(self.h, self.scheme, self.rows, k, self.group)
        return rec

    def apply(self, psi, phi=None, lambdas=None):
        """phi = H psi, complete on every rank (psi must be complete on every rank)."""
        phi = self.h.apply(psi, phi, lambdas)
        return exchange(phi, self.scheme, self.rows, self.group)

    def chebyshev(self, psi, t, e_min, e_max, tol, out=None):
        """exp(-i H t) psi (Eq. 41-44): the library's own driver and O(D) kernels, with this object's
        exchange hook called after every apply (every rank runs the recurrence redundantly on identical
        data, so one exchange per term is all the communication there is)."""
        return self.h.chebyshev(psi, t, e_min, e_max, tol, out)

    def lanczos_bounds(self, psi, m=40, margin=0.05):
        return self.h.lanczos_bounds(psi, m, margin)

    def destroy(self):
        self.h.destroy()
