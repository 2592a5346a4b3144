"""CPU ORACLE for the distributed (multi-GPU) form of phi = H psi -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md P:185-191 (block-row accumulation), P:461-469 (adaptive parallelisation), P:597-618 (row
distribution): "a GPU or GPU group can own a subset of output blocks and accumulate
phi^[n] = sum_m H^[n,m] psi^[m], n in R ... it does not change the Hamiltonian or omit any block
products"; "GPUs in a group are assigned disjoint row sets R_j"; "the local outputs can then be gathered".
The paper fixes neither the row sets nor any other assignment (reading R20), so the oracle states
the two assignments of this build as plain index rules and the contribution of one rank as the definition

    contribution_r[n] = sum_{m : (n,m) owned by r} H^[n,m] psi^[m]           (blocks materialised densely,
                                                                               one numpy matmul per block)

"rows"   rank r owns the contiguous block rows  N r // W <= n < N (r+1) // W  (all m): the paper's
         row-parallel strategy; the contributions have disjoint supports and are GATHERED.
"pairs"  the unordered block pairs {n,m} are dealt round-robin to the ranks in the order
         d = 0, 1, ..., N//2 (circular block distance), n = 0..N-1, m = (n+d) mod N (for 2d = N only
         n < N/2, each pair once); a rank owns both positions (n,m) and (m,n) of its pairs, so a Hermitian
         pair is generated (or stored) once in the whole job; the contributions overlap and are SUMMED.

Pins (tests/test_oracle_partition.py): the ownership masks are disjoint and cover every block, "pairs"
masks are symmetric and balanced to one pair, "rows" masks are row slabs; the contributions of all ranks
add up to the explicit dense matrix product; a "rows" contribution equals the row subset of the full apply
and is zero elsewhere; world = 1 is the plain apply.
"""
from __future__ import annotations

import numpy as np

from . import materialize as _materialize

SCHEMES = ("rows", "pairs")


def owned_blocks(n_blk: int, rank: int, world: int, scheme: str) -> np.ndarray:
    """Boolean mask [n_blk, n_blk]: True where block position (n, m) belongs to `rank`."""
    assert 0 <= rank < world and scheme in SCHEMES
    own = np.zeros((n_blk, n_blk), dtype=bool)
    if scheme == "rows":
        own[n_blk * rank // world: n_blk * (rank + 1) // world, :] = True
        return own
    idx = 0
    for d in range(n_blk // 2 + 1):
        for n in range(n_blk):
            if 2 * d == n_blk and n >= n_blk // 2:
                continue                      # {n, n + N/2} was dealt from the other side
            m = (n + d) % n_blk
            if idx % world == rank:
                own[n, m] = own[m, n] = True
            idx += 1
    return own


def apply_partition(D: int, B: int, seed: int, psi, rank: int, world: int, scheme: str) -> np.ndarray:
    """Contribution of `rank` to phi = H psi: full length D (x k), zero where the rank owns nothing."""
    assert D % B == 0
    n_blk = D // B
    Psi = np.asarray(psi, dtype=np.complex128)
    one = Psi.ndim == 1
    Psi = Psi.reshape(D, -1)
    own = owned_blocks(n_blk, rank, world, scheme)
    out = np.zeros_like(Psi)
    for n in range(n_blk):
        for m in range(n_blk):
            if own[n, m]:
                Hnm = _materialize(D, seed, n * B, B, m * B, B)
                out[n * B:(n + 1) * B] += Hnm @ Psi[m * B:(m + 1) * B]
    return out[:, 0] if one else out


def combine(contributions, scheme: str) -> np.ndarray:
    """The exchange step: every rank ends with the full phi.  Both schemes reduce to a sum because a
    "rows" contribution is zero outside its own rows (the product gathers the segments instead)."""
    assert scheme in SCHEMES
    return np.sum(np.stack(list(contributions)), axis=0)
