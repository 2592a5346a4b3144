"""Seeded synthetic inputs shared by the tests, the oracle legs and bench.py.

This module holds NONE of the method's arithmetic (no Philox4x32, no Box-Muller, no entry rule,
no matvec): it only draws the *inputs* of phi = H psi with numpy's own generator and lists the
five BASELINE.json workloads.  Both the CUDA path and the CPU oracle receive the same arrays.

Recipe: psi has i.i.d. complex standard-normal entries from
``numpy.random.default_rng(seed)``, normalised to unit 2-norm in float64; for complex64 the
normalised vector is rounded to float32 and BOTH sides use the rounded values.  For k vectors
column v is drawn from ``default_rng([seed, v])`` and normalised separately; the layout is
row-major [D][k] (a row of k complex numbers is contiguous).
"""
from __future__ import annotations

import numpy as np

# BASELINE.json configs[0..4] (C1..C5).  "matrix_seed" of C4 and "psi_seed" of C2/C5 are not
# given there; readings R9/R10 fix them to 1234 / 99.
CONFIGS = {
    "C1": dict(D=4096, dtype="c128", B=512, mode="procedural", seed=1234, psi_seed=99, k=1),
    "C2": dict(D=65536, dtype="c128", B=2048, mode="full", seed=1234, psi_seed=99, k=1),
    "C3": dict(D=32768, dtype="c64", B=1024, mode="procedural", seed=8, seed_h0=7, psi_seed=9, k=16),
    "C4": dict(D=262144, dtype="c128", B=4096, mode="procedural", seed=1234, psi_seed=11, k=1),
    "C5": dict(D=131072, dtype="c128", B=4096, mode="partial", seed=21, psi_seed=99, k=1,
               t=50.0, tol=1e-14, e_min=-2.1, e_max=2.1, hbm_budget=150e9),
}


# The same operators from the Hermitian pair cache: side measurements only.
VARIANTS = {
    "C2-pairs": dict(CONFIGS["C2"], mode="pairs"),
    "C5-pairs": dict(CONFIGS["C5"], mode="pairs"),
    # C3's coupling scan with V cached (8.6 GB): each stored block is read once for the 16 vectors
    "C3-cached": dict(CONFIGS["C3"], mode="full"),
    # ... and from the Hermitian pair cache (4.4 GB): the mirrored positions by a second, transposed read
    "C3-pairs": dict(CONFIGS["C3"], mode="pairs"),
    # the same scan in double precision from cached complex128 blocks (17.2 GB): FP64 CUDA-core kernel
    "C3-c128-cached": dict(CONFIGS["C3"], mode="full", dtype="c128"),
}


def make_psi(D: int, seed: int, k: int = 1, dtype: str = "c128") -> np.ndarray:
    """Normalised random complex vector(s): shape [D] for k == 1, else [D, k] row-major."""
    cols = []
    for v in range(k):
        rng = np.random.default_rng(seed if k == 1 else [seed, v])
        x = rng.standard_normal(D) + 1j * rng.standard_normal(D)
        cols.append(x / np.linalg.norm(x))
    psi = cols[0] if k == 1 else np.ascontiguousarray(np.stack(cols, axis=1))
    if dtype == "c64":
        psi = psi.astype(np.complex64)
    return psi


def lambda_grid(k: int, lo: float = 0.0, hi: float = 2.0) -> np.ndarray:
    """k coupling strengths evenly spaced in [lo, hi], both endpoints included (configs[2])."""
    if k == 1:
        return np.array([hi], dtype=np.float64)
    return lo + (hi - lo) * np.arange(k, dtype=np.float64) / (k - 1)


def sample_rows(D: int, n: int, seed: int = 0) -> np.ndarray:
    """Row sample for full-size parity: both ends, block edges and n random rows, sorted."""
    rng = np.random.default_rng([D, seed])
    fixed = np.array([0, 1, D // 2 - 1, D // 2, D - 2, D - 1], dtype=np.int64)
    rand = rng.integers(0, D, size=n, dtype=np.int64)
    return np.unique(np.concatenate([fixed, rand]))


def stratified_rows(D: int, B: int, n_min: int = 8192, tile: int = 128) -> np.ndarray:
    """Row sample for full-size parity that provably covers the kernels' decomposition: every `tile`-row tile of the
    operator contributes S = ceil(n_min / (D / tile)) rows at residues (37 t + s * (tile // S)) mod tile (t = tile
    index, s = 0..S-1), so every tile, hence every block row, every residue mod `tile` (every (lane, row-in-lane)
    position of a 32 x 4 row tile) and every warp's strip is hit; plus the first and last row of every block.  Sorted,
    unique, deterministic (no random numbers)."""
    n_tiles = D // tile
    S = min(tile, max(1, -(-n_min // n_tiles)))
    t = np.arange(n_tiles, dtype=np.int64)[:, None]
    s = np.arange(S, dtype=np.int64)[None, :]
    rows = (t * tile + (37 * t + s * (tile // S)) % tile).ravel()
    blocks = np.arange(D // B, dtype=np.int64) * B
    return np.unique(np.concatenate([rows, blocks, blocks + B - 1]))


def dense_matrix(D: int, seed: int, hermitian: bool = True) -> np.ndarray:
    """Seeded dense D x D complex matrix with O(1/sqrt(D)) entries: the externally stored operator of the Eq. 10
    tests (an input of the method, not part of its arithmetic)."""
    rng = np.random.default_rng([seed, D, 10])
    M = (rng.standard_normal((D, D)) + 1j * rng.standard_normal((D, D))) / np.sqrt(2.0 * D)
    return (M + M.conj().T) / np.sqrt(2.0) if hermitian else M


def small_hermitian(d: int, seed: int) -> np.ndarray:
    """Seeded d x d Hermitian matrix with O(1) entries (system-side operators H_S, A of the system-bath
    workload; an input of the method, not part of its arithmetic)."""
    rng = np.random.default_rng([seed, d])
    M = rng.standard_normal((d, d)) + 1j * rng.standard_normal((d, d))
    return (M + M.conj().T) / 2.0


# The paper's own run: 18 qubits, d_S = 4, d_B = 65536, complex64, two cached dense
# bath-side operators (H_B, B_1) applied to R = 4 columns, N_blk = 16 (b = 4096).  Operators synthetic (R19).
SYSTEM_BATH = dict(d_B=65536, d_S=4, B=4096, dtype="c64", seed_HB=31, seed_B1=32, seed_HS=33, seed_A=34,
                   g=0.5, psi_seed=35, mode="full", paper_seconds_per_apply=0.104089,
                   paper_hardware="2 x NVIDIA L40S (one row group), CuPy, complex64 (P:771-775)")
