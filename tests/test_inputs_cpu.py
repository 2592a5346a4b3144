"""The seeded input generators and row samples (paper_2606_31598_b200/inputs.py hold no method arithmetic; these
tests pin the properties the full-size parity tests rely on)."""
import numpy as np

from paper_2606_31598_b200.inputs import CONFIGS, SYSTEM_BATH, make_psi, stratified_rows


def test_stratified_rows_cover_every_tile_residue_block_and_block_edge():
    shapes = [(c["D"], c["B"]) for c in CONFIGS.values()] + [(SYSTEM_BATH["d_B"], SYSTEM_BATH["B"]), (32768, 4096)]
    for D, B in shapes:
        rows = stratified_rows(D, B)
        assert rows.dtype == np.int64 and np.all(np.diff(rows) > 0) and rows[0] == 0 and rows[-1] == D - 1
        assert len(rows) >= min(D, 8192)
        assert set(rows // 128) == set(range(D // 128))            # every 128-row tile (every CTA strip of every kernel)
        assert set(rows % 128) == set(range(128))                  # every (lane, row-in-lane) position of a 32 x 4 tile
        assert set(rows // B) == set(range(D // B))                # every block row
        edges = np.arange(D // B) * B
        assert np.all(np.isin(edges, rows)) and np.all(np.isin(edges + B - 1, rows))
        # within one 128-row tile the sampled residues are spread over the four 32-row groups (the rows of one lane)
        if D // 128 <= 2048:
            t0 = rows[rows // 128 == 5] % 128
            assert len(set(t0 // 32)) >= min(4, len(t0))
    assert np.array_equal(stratified_rows(4096, 512), np.arange(4096))   # small D: all rows


def test_make_psi_is_normalised_seeded_and_column_independent():
    a = make_psi(4096, 99)
    assert abs(np.linalg.norm(a) - 1.0) < 1e-14 and np.array_equal(a, make_psi(4096, 99))
    P = make_psi(1024, 9, k=4, dtype="c64")
    assert P.shape == (1024, 4) and P.dtype == np.complex64 and P.flags["C_CONTIGUOUS"]
    assert np.allclose(np.linalg.norm(P.astype(np.complex128), axis=0), 1.0, atol=1e-6)
    assert not np.allclose(P[:, 0], P[:, 1])
