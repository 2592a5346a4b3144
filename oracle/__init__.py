"""CPU ORACLE for phi = H psi -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2606_31598_b200`` (the CUDA path) and never imports it.

``mfh_oracle.c`` holds the arithmetic of the matvec (Philox4x32-10, Box-Muller, the GUE entry
rule, the two-level loop of PAPER.md Eq. 5/7); this module is the ctypes marshalling around it
plus the Chebyshev propagator (``chebyshev.py``), which follows PAPER.md Eq. 41-44 step by step.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mfh_oracle.c")
_LIB = os.path.join(_HERE, "libmfh_oracle.so")

_lib = None


def build(force: bool = False) -> str:
    """Compile mfh_oracle.c with gcc (-O2, no FMA contraction, OpenMP over rows)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11",
               _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        u32p = ctypes.POINTER(ctypes.c_uint32)
        f64p = ctypes.POINTER(ctypes.c_double)
        i64p = ctypes.POINTER(ctypes.c_int64)
        i64, u64, u32 = ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint32
        L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.orc_philox4x32_10.restype = None
        L.orc_philox_pairs.argtypes = [u64, u32, u32p, u32p, i64, u32p]
        L.orc_philox_pairs.restype = None
        L.orc_uniform.argtypes = [u32]
        L.orc_uniform.restype = ctypes.c_double
        L.orc_box_muller.argtypes = [ctypes.c_double, ctypes.c_double, f64p, f64p]
        L.orc_box_muller.restype = None
        L.orc_entry.argtypes = [i64, u64, i64, i64, f64p, f64p]
        L.orc_entry.restype = None
        L.orc_materialize.argtypes = [i64, u64, i64, i64, i64, i64, f64p]
        L.orc_materialize.restype = None
        L.orc_h0.argtypes = [i64, u64, f64p]
        L.orc_h0.restype = None
        L.orc_apply_rows.argtypes = [i64, i64, u64, i64, f64p, i64p, i64, f64p]
        L.orc_apply_rows.restype = None
        L.orc_apply_scan_rows.argtypes = [i64, i64, u64, u64, i64, f64p, f64p, i64p, i64, f64p]
        L.orc_apply_scan_rows.restype = None
        L.orc_num_threads.argtypes = []
        L.orc_num_threads.restype = ctypes.c_int
        _lib = L
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


def num_threads() -> int:
    return int(lib().orc_num_threads())


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.empty(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c, ctypes.c_uint32), _p(k, ctypes.c_uint32), _p(out, ctypes.c_uint32))
    return out


def philox_pairs(seed: int, stream: int, i, j) -> np.ndarray:
    """Raw words for ctr=(min(i,j), max(i,j), stream, 0), key=seed; shape [n, 4]."""
    i = np.ascontiguousarray(i, dtype=np.uint32)
    j = np.ascontiguousarray(j, dtype=np.uint32)
    out = np.empty((i.size, 4), dtype=np.uint32)
    lib().orc_philox_pairs(seed, stream, _p(i, ctypes.c_uint32), _p(j, ctypes.c_uint32), i.size,
                           _p(out, ctypes.c_uint32))
    return out


def uniform(x: int) -> float:
    return float(lib().orc_uniform(int(x)))


def box_muller(u1: float, u2: float):
    g1, g2 = ctypes.c_double(), ctypes.c_double()
    lib().orc_box_muller(u1, u2, ctypes.byref(g1), ctypes.byref(g2))
    return g1.value, g2.value


def entry(D: int, seed: int, i: int, j: int) -> complex:
    re, im = ctypes.c_double(), ctypes.c_double()
    lib().orc_entry(D, seed, i, j, ctypes.byref(re), ctypes.byref(im))
    return complex(re.value, im.value)


def materialize(D: int, seed: int, i0: int = 0, ni: int | None = None, j0: int = 0,
                nj: int | None = None) -> np.ndarray:
    """Dense H[i0:i0+ni, j0:j0+nj] as complex128."""
    ni = D - i0 if ni is None else ni
    nj = D - j0 if nj is None else nj
    out = np.empty((ni, nj), dtype=np.complex128)
    lib().orc_materialize(D, seed, i0, ni, j0, nj, _p(out, ctypes.c_double))
    return out


def h0_diagonal(D: int, seed_h0: int) -> np.ndarray:
    out = np.empty(D, dtype=np.float64)
    lib().orc_h0(D, seed_h0, _p(out, ctypes.c_double))
    return out


def _as_Psi(psi, D):
    Psi = np.ascontiguousarray(psi, dtype=np.complex128)
    if Psi.ndim == 1:
        Psi = Psi.reshape(D, 1)
    assert Psi.shape[0] == D and Psi.shape[1] <= 64
    return Psi


def apply(D: int, B: int, seed: int, psi, rows=None) -> np.ndarray:
    """phi = H psi by the block loop of Eq. 7.  psi: [D] or [D,k] (any complex dtype; evaluated
    in double).  rows: optional subset of output rows (full-size parity samples)."""
    assert D % B == 0
    Psi = _as_Psi(psi, D)
    k = Psi.shape[1]
    if rows is None:
        nrows, rp = D, None
    else:
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        nrows, rp = rows.size, _p(rows, ctypes.c_int64)
    out = np.empty((nrows, k), dtype=np.complex128)
    lib().orc_apply_rows(D, B, seed, k, _p(Psi, ctypes.c_double), rp, nrows, _p(out, ctypes.c_double))
    return out[:, 0] if np.ndim(psi) == 1 else out


def apply_scan(D: int, B: int, seed_v: int, seed_h0: int, lambdas, Psi, rows=None) -> np.ndarray:
    """Phi[:,v] = h0 (.) Psi[:,v] + lambda_v V Psi[:,v]  (BASELINE.json configs[2])."""
    assert D % B == 0
    Psi = _as_Psi(Psi, D)
    k = Psi.shape[1]
    lam = np.ascontiguousarray(lambdas, dtype=np.float64)
    assert lam.size == k
    if rows is None:
        nrows, rp = D, None
    else:
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        nrows, rp = rows.size, _p(rows, ctypes.c_int64)
    out = np.empty((nrows, k), dtype=np.complex128)
    lib().orc_apply_scan_rows(D, B, seed_v, seed_h0, k, _p(lam, ctypes.c_double),
                              _p(Psi, ctypes.c_double), rp, nrows, _p(out, ctypes.c_double))
    return out


from .chebyshev import (bessel_i_scaled_table, bessel_j_table, chebyshev_imag_n_terms, chebyshev_imag_propagate,  # noqa: E402,F401
                        chebyshev_n_terms, chebyshev_propagate)
from .lanczos import lanczos_bounds, lanczos_tridiagonal, ritz_extremes  # noqa: E402,F401
from .system_bath import sb_apply  # noqa: E402,F401
from .partition import apply_partition, combine as combine_partition, owned_blocks  # noqa: E402,F401
from .analytic import analytic_apply, analytic_matrix, theta_array  # noqa: E402,F401
from .external import block_apply, stored_blocks  # noqa: E402,F401
from . import surrogate  # noqa: E402,F401
