"""Pins of the distributed-execution oracle (oracle/partition.py; PAPER.md P:185-191, P:461-469,
P:597-618; R20)."""
import numpy as np
import pytest

import oracle
from paper_2606_31598_b200.inputs import make_psi

D, B, SEED = 256, 32, 1234     # 8 x 8 blocks


@pytest.mark.parametrize("scheme", ["rows", "pairs"])
@pytest.mark.parametrize("n_blk,world", [(8, 1), (8, 2), (8, 3), (8, 8), (7, 2), (16, 5), (64, 8), (2, 2)])
def test_masks_are_a_disjoint_cover(scheme, n_blk, world):
    masks = [oracle.owned_blocks(n_blk, r, world, scheme) for r in range(world)]
    total = np.sum(np.stack(masks).astype(int), axis=0)
    assert np.array_equal(total, np.ones((n_blk, n_blk), dtype=int))      # every block exactly once


@pytest.mark.parametrize("n_blk,world", [(8, 2), (8, 3), (16, 5), (64, 8), (7, 2)])
def test_pairs_masks_are_symmetric_and_balanced(n_blk, world):
    counts = []
    for r in range(world):
        own = oracle.owned_blocks(n_blk, r, world, "pairs")
        assert np.array_equal(own, own.T)                                 # a pair lives on ONE rank
        counts.append(int(np.triu(own).sum()))                            # unordered pairs incl. diagonal
    assert sum(counts) == n_blk * (n_blk + 1) // 2
    assert max(counts) - min(counts) <= 1


def test_rows_masks_are_contiguous_row_slabs():
    for n_blk, world in [(8, 2), (8, 3), (16, 5)]:
        edges = [n_blk * r // world for r in range(world + 1)]
        for r in range(world):
            own = oracle.owned_blocks(n_blk, r, world, "rows")
            rows = np.flatnonzero(own.any(axis=1))
            assert np.array_equal(rows, np.arange(edges[r], edges[r + 1]))
            assert own[rows].all()                                        # whole block rows


@pytest.mark.parametrize("scheme", ["rows", "pairs"])
@pytest.mark.parametrize("world", [1, 2, 3, 8])
def test_contributions_add_up_to_the_dense_product(scheme, world):
    psi = make_psi(D, 99)
    ref = oracle.materialize(D, SEED) @ psi                               # explicit dense matrix (pinned elsewhere)
    parts = [oracle.apply_partition(D, B, SEED, psi, r, world, scheme) for r in range(world)]
    phi = oracle.combine_partition(parts, scheme)
    assert np.linalg.norm(phi - ref) <= 1e-13 * np.linalg.norm(ref)
    if world > 1:                                                         # no rank does all the work
        assert all(np.linalg.norm(p - ref) > 1e-3 for p in parts)


def test_rows_contribution_is_the_row_subset_of_the_full_apply():
    psi = make_psi(D, 99)
    world = 3
    n_blk = D // B
    for r in range(world):
        part = oracle.apply_partition(D, B, SEED, psi, r, world, "rows")
        lo, hi = B * (n_blk * r // world), B * (n_blk * (r + 1) // world)
        ref = oracle.apply(D, B, SEED, psi, rows=np.arange(lo, hi))
        assert np.linalg.norm(part[lo:hi] - ref) <= 1e-13 * np.linalg.norm(ref)
        assert not part[:lo].any() and not part[hi:].any()                # disjoint supports: gather == sum


def test_world_one_is_the_plain_apply_and_k_vectors():
    Psi = make_psi(D, 9, k=4)
    ref = oracle.apply(D, B, SEED, Psi)
    for scheme in ("rows", "pairs"):
        assert np.allclose(oracle.apply_partition(D, B, SEED, Psi, 0, 1, scheme), ref, rtol=0, atol=1e-14)
    parts = [oracle.apply_partition(D, B, SEED, Psi, r, 2, "pairs") for r in range(2)]
    assert np.allclose(oracle.combine_partition(parts, "pairs"), ref, rtol=0, atol=1e-14)
