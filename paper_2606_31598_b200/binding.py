"""Thin ctypes binding of include/mfh.h -- argument marshalling only.

Every step of phi = H psi runs in the CUDA kernels of ``lib/libmfh.so``; this module converts
torch tensors to device pointers and the current torch stream to a ``cudaStream_t``.  There is no
CPU fallback: loading fails loudly when the library is missing, and every compute call needs a
CUDA device.  PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
import json
import os

from . import build as _build

MFH_OK = 0
MFH_ERR_INVALID_ARG, MFH_ERR_BAD_STATE, MFH_ERR_OUT_OF_MEMORY = 1, 2, 3
MFH_ERR_CUDA, MFH_ERR_NOT_CONVERGED, MFH_ERR_UNSUPPORTED = 4, 5, 6
MFH_C128, MFH_C64 = 0, 1
MFH_SRC_GUE, MFH_SRC_DIAG_PLUS_GUE, MFH_SRC_ANALYTIC, MFH_SRC_EXTERNAL = 0, 1, 2, 3
SOURCES = {"gue": MFH_SRC_GUE, "diag_plus_gue": MFH_SRC_DIAG_PLUS_GUE, "analytic": MFH_SRC_ANALYTIC,
           "external": MFH_SRC_EXTERNAL}
MFH_MODE_AUTO, MFH_MODE_PROCEDURAL, MFH_MODE_PARTIAL, MFH_MODE_FULL, MFH_MODE_PAIRS = 0, 1, 2, 3, 4
MFH_MAX_K = 16
MFH_PART_NONE, MFH_PART_ROWS, MFH_PART_PAIRS = 0, 1, 2
PARTITIONS = {"none": MFH_PART_NONE, "rows": MFH_PART_ROWS, "pairs": MFH_PART_PAIRS}

DTYPES = {"c128": MFH_C128, "c64": MFH_C64}
MODES = {"auto": MFH_MODE_AUTO, "procedural": MFH_MODE_PROCEDURAL, "partial": MFH_MODE_PARTIAL,
         "full": MFH_MODE_FULL, "pairs": MFH_MODE_PAIRS}

# every symbol include/mfh.h declares (tests check that the library exports all of them)
SYMBOLS = ["mfh_create", "mfh_plan_analytic", "mfh_plan_node_analytic", "mfh_plan", "mfh_apply", "mfh_apply_host", "mfh_apply_timed", "mfh_timing_begin", "mfh_timing_end",
           "mfh_chebyshev", "mfh_chebyshev_imag", "mfh_chebyshev_scan", "mfh_chebyshev_steps", "mfh_lanczos_bounds", "mfh_destroy", "mfh_last_error", "mfh_get_plan", "mfh_debug_philox",
           "mfh_materialize_block", "mfh_debug_h0", "mfh_debug_bessel_j", "mfh_debug_poison", "mfh_debug_selfcheck", "mfh_debug_corrupt_guard", "mfh_debug_pipe_rates", "mfh_sb_create", "mfh_sb_plan", "mfh_sb_apply",
           "mfh_sb_destroy", "mfh_set_partition", "mfh_get_partition_rows", "mfh_set_exchange", "mfh_debug_read_bandwidth", "mfh_set_source_params", "mfh_set_block", "mfh_surrogate_theta_size", "mfh_surrogate_fit",
           "mfh_surrogate_predict", "mfh_surrogate_loss_grad", "mfh_surrogate_features", "mfh_plan_hybrid", "mfh_apply_static"]

_lib = None


class MfhError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"mfh error {code}: {msg}")
        self.code = code


def lib():
    """Load lib/libmfh.so (must have been built: ``python -m paper_2606_31598_b200.build``)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: build the CUDA library first "
                           "(python paper_2606_31598_b200/build.py); there is no CPU fallback")
    L = ctypes.CDLL(path)
    vp, i32, i64, u32, u64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_uint32, ctypes.c_uint64
    dbl, cp, sz = ctypes.c_double, ctypes.c_char_p, ctypes.c_size_t
    L.mfh_create.argtypes = [ctypes.POINTER(vp), i64, i32, u64, i32, dbl, i32, u64]
    L.mfh_plan_analytic.argtypes = [i64, i32, i32, i32, i32, i64, i64, cp, sz]
    L.mfh_plan_node_analytic.argtypes = [i64, i32, i32, i32, i64, i32, i64, i32, i32, i32, i64, cp, sz]
    L.mfh_plan.argtypes = [vp, i32, i32, i64, i64, i32, vp, cp, sz]
    L.mfh_apply.argtypes = [vp, vp, vp, i32, ctypes.POINTER(dbl), vp]
    L.mfh_apply_host.argtypes = [vp, vp, vp, i32, ctypes.POINTER(dbl), vp]
    L.mfh_apply_static.argtypes = [i64, u64, dbl, vp, vp, vp]
    L.mfh_apply_timed.argtypes = [vp, vp, vp, i32, ctypes.POINTER(dbl), vp, ctypes.POINTER(ctypes.c_float)]
    L.mfh_timing_begin.argtypes = [vp, i32]
    L.mfh_timing_end.argtypes = [vp, ctypes.POINTER(ctypes.c_float), ctypes.POINTER(i32), vp]
    L.mfh_chebyshev.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, ctypes.POINTER(i32), vp]
    L.mfh_chebyshev_scan.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, ctypes.POINTER(dbl), ctypes.POINTER(i32), vp]
    L.mfh_chebyshev_imag.argtypes = [vp, vp, vp, dbl, dbl, dbl, dbl, ctypes.POINTER(i32), vp]
    L.mfh_chebyshev_steps.argtypes = [vp, vp, vp, dbl, i32, dbl, dbl, dbl, ctypes.POINTER(i32), vp]
    L.mfh_lanczos_bounds.argtypes = [vp, vp, i32, dbl, ctypes.POINTER(dbl), ctypes.POINTER(dbl), ctypes.POINTER(dbl),
                                     ctypes.POINTER(dbl), vp]
    L.mfh_set_partition.argtypes = [vp, i32, i32, i32]
    L.mfh_set_exchange.argtypes = [vp, vp, vp]
    L.mfh_set_source_params.argtypes = [vp, ctypes.POINTER(dbl)]
    L.mfh_set_block.argtypes = [vp, i32, i32, vp, i32, vp]
    L.mfh_get_partition_rows.argtypes = [vp, ctypes.POINTER(i32), ctypes.POINTER(i32), ctypes.POINTER(i32)]
    L.mfh_destroy.argtypes = [vp]
    L.mfh_last_error.argtypes = []
    L.mfh_last_error.restype = cp
    L.mfh_get_plan.argtypes = [vp, cp, sz]
    L.mfh_debug_philox.argtypes = [u64, u32, vp, vp, i64, vp, vp]
    L.mfh_materialize_block.argtypes = [vp, i32, i32, vp, vp]
    L.mfh_debug_h0.argtypes = [vp, vp, vp]
    L.mfh_debug_poison.argtypes = [vp, vp]
    L.mfh_debug_corrupt_guard.argtypes = [vp, i32, i32]
    L.mfh_debug_selfcheck.argtypes = [vp, ctypes.POINTER(i64), vp]
    L.mfh_debug_bessel_j.argtypes = [dbl, i32, ctypes.POINTER(dbl)]
    L.mfh_debug_pipe_rates.argtypes = [i32, ctypes.POINTER(dbl), vp]
    L.mfh_debug_read_bandwidth.argtypes = [vp, sz, ctypes.POINTER(dbl), vp]
    L.mfh_sb_create.argtypes = [ctypes.POINTER(vp), i64, i32, i32, u64, u64, i32, vp, vp, dbl]
    L.mfh_sb_plan.argtypes = [vp, i32, i64, i64, vp, cp, sz]
    L.mfh_sb_apply.argtypes = [vp, vp, vp, vp]
    L.mfh_sb_destroy.argtypes = [vp]
    for name in SYMBOLS:
        if name not in ("mfh_last_error", "mfh_surrogate_theta_size"):
            getattr(L, name).restype = ctypes.c_int
    _lib = L
    return L


def _check(rc: int):
    if rc != MFH_OK:
        raise MfhError(rc, lib().mfh_last_error().decode())


def _stream():
    import torch
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _lam(lambdas, k):
    if lambdas is None:
        return None
    arr = (ctypes.c_double * k)(*[float(x) for x in lambdas])
    return arr


def plan_analytic(D: int, dtype: str, k: int = 1, mode: str = "auto", B: int = 0,
                  n_applies_hint: int = 1, hbm_free_bytes: int = 180 * 10**9) -> dict:
    """Host-only analytic planner (Algorithm 1); needs no GPU."""
    buf = ctypes.create_string_buffer(1 << 16)
    rc = lib().mfh_plan_analytic(D, DTYPES[dtype], k, MODES[mode], B, n_applies_hint, hbm_free_bytes,
                                 buf, len(buf))
    rec = json.loads(buf.value.decode()) if buf.value else {}
    if rc != MFH_OK:
        raise MfhError(rc, lib().mfh_last_error().decode())
    return rec


def plan_node_analytic(D: int, dtype: str, k: int, n_op: int, n_tasks: int, n_gpus: int, hbm_free_bytes_per_gpu: int,
                       mode: str = "auto", B: int = 0, scheme: str = "pairs", n_applies_per_task: int = 1) -> dict:
    """Host-only node-level planner: row-group size, GPU groups and task waves (Eq. 19); needs no GPU."""
    buf = ctypes.create_string_buffer(1 << 16)
    rc = lib().mfh_plan_node_analytic(D, DTYPES[dtype], k, n_op, n_tasks, n_gpus, int(hbm_free_bytes_per_gpu), MODES[mode], B,
                                      PARTITIONS[scheme], n_applies_per_task, buf, len(buf))
    rec = json.loads(buf.value.decode()) if buf.value else {}
    if rc != MFH_OK:
        raise MfhError(rc, lib().mfh_last_error().decode())
    return rec


class Hamiltonian:
    """Handle of one seeded Hamiltonian (mfh_create ... mfh_destroy)."""

    def __init__(self, D: int, B: int = 0, seed: int = 0, dtype: str = "c128", kind: str = "gue",
                 lam: float = 1.0, seed_h0: int = 0):
        self.D, self.dtype, self.k = D, dtype, None
        self._h = ctypes.c_void_p()
        _check(lib().mfh_create(ctypes.byref(self._h), D, B, seed, SOURCES[kind], lam, DTYPES[dtype], seed_h0))

    # -- torch plumbing ---------------------------------------------------------------------
    def _torch_dtype(self):
        import torch
        return torch.complex128 if self.dtype == "c128" else torch.complex64

    def _check_vec(self, x, k):
        assert x.is_cuda and x.is_contiguous() and x.dtype == self._torch_dtype()
        assert x.numel() == self.D * k, (x.shape, self.D, k)

    # -- C ABI ------------------------------------------------------------------------------
    def plan(self, mode: str = "auto", k: int = 1, n_applies_hint: int = 1, hbm_budget_bytes: int = 0,
             measure: bool = False) -> dict:
        buf = ctypes.create_string_buffer(1 << 16)
        _check(lib().mfh_plan(self._h, MODES[mode], k, n_applies_hint, int(hbm_budget_bytes),
                              1 if measure else 0, _stream(), buf, len(buf)))
        self.k = k
        return json.loads(buf.value.decode())

    def set_source_params(self, theta):
        """Parameters (t, alpha, phi, W, beta, delta) of the analytic source (kind="analytic"); call before plan."""
        arr = (ctypes.c_double * 6)(*[float(x) for x in theta])
        _check(lib().mfh_set_source_params(self._h, arr))

    def set_block(self, n: int, m: int, block):
        """Supply the stored block (n, m) of an external operator (kind="external"): a B x B complex torch tensor
        (device or host) or numpy array of the handle's dtype, row-major."""
        import numpy as np
        if isinstance(block, np.ndarray):
            want = np.complex128 if self.dtype == "c128" else np.complex64
            arr = np.ascontiguousarray(block, dtype=want)
            _check(lib().mfh_set_block(self._h, n, m, arr.ctypes.data, 0, _stream()))
        else:
            assert block.is_contiguous() and block.dtype == self._torch_dtype()
            _check(lib().mfh_set_block(self._h, n, m, block.data_ptr(), 1 if block.is_cuda else 0, _stream()))

    def set_partition(self, rank: int, world: int, scheme: str = "pairs"):
        """Distributed execution: this handle computes rank `rank`'s share of phi (call before plan)."""
        _check(lib().mfh_set_partition(self._h, rank, world, PARTITIONS[scheme]))

    def partition_rows(self):
        """(first row, number of rows) of phi that apply() writes on this handle."""
        a, b, c = ctypes.c_int32(0), ctypes.c_int32(0), ctypes.c_int32(0)
        _check(lib().mfh_get_partition_rows(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
        return a.value * c.value, b.value * c.value

    def get_plan(self) -> dict:
        buf = ctypes.create_string_buffer(4096)
        _check(lib().mfh_get_plan(self._h, buf, len(buf)))
        return json.loads(buf.value.decode())

    def apply(self, psi, phi=None, lambdas=None):
        """phi = H psi on device tensors ([D] or [D,k] complex), asynchronous on the current stream."""
        import torch
        k = self.k or 1
        self._check_vec(psi, k)
        if phi is None:
            phi = torch.empty_like(psi)
        self._check_vec(phi, k)
        _check(lib().mfh_apply(self._h, psi.data_ptr(), phi.data_ptr(), k, _lam(lambdas, k), _stream()))
        return phi

    def apply_timed(self, psi, phi, lambdas=None) -> dict:
        """One apply with CUDA events around each launch; returns milliseconds per kernel."""
        k = self.k or 1
        self._check_vec(psi, k)
        self._check_vec(phi, k)
        ms = (ctypes.c_float * 4)()
        _check(lib().mfh_apply_timed(self._h, psi.data_ptr(), phi.data_ptr(), k, _lam(lambdas, k),
                                     _stream(), ms))
        return {"cached": ms[0], "procedural": ms[1], "reduce": ms[2], "total": ms[3]}

    def timing_begin(self, n_applies: int):
        """Arm in-pass per-kernel timing for the next n_applies apply() calls (no synchronisation inside the pass)."""
        self._timing_n = int(n_applies)
        _check(lib().mfh_timing_begin(self._h, self._timing_n))

    def timing_end(self):
        """Synchronise and return one dict of milliseconds per recorded apply (keys as apply_timed)."""
        ms = (ctypes.c_float * (4 * self._timing_n))()
        n = ctypes.c_int32(0)
        _check(lib().mfh_timing_end(self._h, ms, ctypes.byref(n), _stream()))
        return [{"cached": ms[4 * a], "procedural": ms[4 * a + 1], "reduce": ms[4 * a + 2], "total": ms[4 * a + 3]}
                for a in range(n.value)]

    def apply_host(self, psi_host, phi_host, lambdas=None):
        """End-to-end call with HOST (pinned) torch tensors; synchronises."""
        k = self.k or 1
        assert not psi_host.is_cuda and not phi_host.is_cuda
        _check(lib().mfh_apply_host(self._h, psi_host.data_ptr(), phi_host.data_ptr(), k,
                                    _lam(lambdas, k), _stream()))
        return phi_host

    def chebyshev(self, psi, t: float, e_min: float, e_max: float, tol: float, out=None):
        import torch
        self._check_vec(psi, 1)
        if out is None:
            out = torch.empty_like(psi)
        n = ctypes.c_int32(0)
        _check(lib().mfh_chebyshev(self._h, psi.data_ptr(), out.data_ptr(), t, e_min, e_max, tol,
                                   ctypes.byref(n), _stream()))
        return out, int(n.value)

    def chebyshev_scan(self, psi, t: float, e_min: float, e_max: float, tol: float, lambdas=None, out=None):
        """out[:, v] = exp(-i H_v t) psi[:, v] for the k columns of a k-vector plan; returns (out, n_terms)."""
        import torch
        k = self.k or 1
        self._check_vec(psi, k)
        if out is None:
            out = torch.empty_like(psi)
        n = ctypes.c_int32(0)
        _check(lib().mfh_chebyshev_scan(self._h, psi.data_ptr(), out.data_ptr(), t, e_min, e_max, tol, _lam(lambdas, k),
                                        ctypes.byref(n), _stream()))
        return out, int(n.value)

    def chebyshev_imag(self, psi, beta: float, e_min: float, e_max: float, tol: float, out=None):
        """out = exp(-beta (H - e_min)) psi (imaginary-time filter); returns (out, n_terms)."""
        import torch
        self._check_vec(psi, 1)
        if out is None:
            out = torch.empty_like(psi)
        n = ctypes.c_int32(0)
        _check(lib().mfh_chebyshev_imag(self._h, psi.data_ptr(), out.data_ptr(), beta, e_min, e_max, tol,
                                        ctypes.byref(n), _stream()))
        return out, int(n.value)

    def chebyshev_steps(self, psi, tau: float, n_steps: int, e_min: float, e_max: float, tol: float, out=None):
        import torch
        self._check_vec(psi, 1)
        if out is None:
            out = torch.empty_like(psi)
        n = ctypes.c_int32(0)
        _check(lib().mfh_chebyshev_steps(self._h, psi.data_ptr(), out.data_ptr(), tau, n_steps, e_min, e_max, tol,
                                         ctypes.byref(n), _stream()))
        return out, int(n.value)

    def lanczos_bounds(self, psi, m: int = 40, margin: float = 0.05):
        """(e_min, e_max, alpha[m], beta[m]) from m matrix-free Lanczos steps started at psi."""
        import numpy as np
        self._check_vec(psi, 1)
        mm = min(m, self.D)
        e0, e1 = ctypes.c_double(0.0), ctypes.c_double(0.0)
        alpha = (ctypes.c_double * mm)()
        beta = (ctypes.c_double * mm)()
        _check(lib().mfh_lanczos_bounds(self._h, psi.data_ptr(), m, margin, ctypes.byref(e0), ctypes.byref(e1),
                                        alpha, beta, _stream()))
        return float(e0.value), float(e1.value), np.array(alpha[:]), np.array(beta[:])

    def materialize_block(self, n: int, m: int, B: int):
        import torch
        out = torch.empty((B, B), dtype=self._torch_dtype(), device="cuda")
        _check(lib().mfh_materialize_block(self._h, n, m, out.data_ptr(), _stream()))
        return out

    def h0(self):
        import torch
        out = torch.empty(self.D, dtype=torch.float64 if self.dtype == "c128" else torch.float32,
                          device="cuda")
        _check(lib().mfh_debug_h0(self._h, out.data_ptr(), _stream()))
        return out

    def debug_poison(self):
        """Fill the library's partial-sum workspace and Chebyshev scratch with NaN (self-check: stale reads)."""
        _check(lib().mfh_debug_poison(self._h, _stream()))

    def debug_selfcheck(self) -> int:
        """Number of corrupted guard-band bytes around the library-owned buffers (0 = no out-of-bounds write)."""
        bad = ctypes.c_int64(-1)
        _check(lib().mfh_debug_selfcheck(self._h, ctypes.byref(bad), _stream()))
        return int(bad.value)

    def destroy(self):
        if self._h:
            lib().mfh_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


class SystemBath:
    """H = H_S (x) I + I (x) H_B + g A (x) B_1 on X[d_B][d_S] (mfh_sb_create ... mfh_sb_destroy)."""

    def __init__(self, d_B: int, d_S: int, B: int, seed_HB: int, seed_B1: int, H_S, A, g: float, dtype: str = "c64"):
        import numpy as np
        self.d_B, self.d_S, self.dtype = d_B, d_S, dtype
        hs = np.ascontiguousarray(H_S, dtype=np.complex128)
        a = np.ascontiguousarray(A, dtype=np.complex128)
        assert hs.shape == (d_S, d_S) and a.shape == (d_S, d_S)
        self._h = ctypes.c_void_p()
        _check(lib().mfh_sb_create(ctypes.byref(self._h), d_B, d_S, B, seed_HB, seed_B1, DTYPES[dtype],
                                   hs.ctypes.data, a.ctypes.data, float(g)))

    def plan(self, mode: str = "auto", n_applies_hint: int = 1, hbm_budget_bytes: int = 0) -> dict:
        buf = ctypes.create_string_buffer(1 << 14)
        _check(lib().mfh_sb_plan(self._h, MODES[mode], n_applies_hint, int(hbm_budget_bytes), _stream(), buf, len(buf)))
        return json.loads(buf.value.decode())

    def apply(self, X, Y=None):
        import torch
        want = torch.complex128 if self.dtype == "c128" else torch.complex64
        assert X.is_cuda and X.is_contiguous() and X.dtype == want and X.numel() == self.d_B * self.d_S
        if Y is None:
            Y = torch.empty_like(X)
        _check(lib().mfh_sb_apply(self._h, X.data_ptr(), Y.data_ptr(), _stream()))
        return Y

    def destroy(self):
        if self._h:
            lib().mfh_sb_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


STATIC_MAX_D = 16384   # include/mfh.h MFH_STATIC_MAX_D


def apply_static(D: int, seed: int, lam: float, psi, phi=None):
    """phi = lam * V(seed) psi through mfh_apply_static: no handle, no plan, no allocation inside the library (the
    output tensor is the caller's; one is made here only when none is passed).  complex128, one vector, D <= STATIC_MAX_D."""
    import torch
    assert psi.is_cuda and psi.dtype == torch.complex128 and psi.is_contiguous() and psi.numel() == D
    if phi is None:
        phi = torch.empty_like(psi)
    assert phi.is_cuda and phi.dtype == torch.complex128 and phi.is_contiguous() and phi.numel() == D
    _check(lib().mfh_apply_static(int(D), int(seed), float(lam), psi.data_ptr(), phi.data_ptr(), _stream()))
    return phi


def debug_philox(seed: int, stream_id: int, i, j):
    """Raw Philox4x32-10 words [n,4] (uint32 as int64-safe torch.int32 bit patterns) for index pairs."""
    import torch
    assert i.is_cuda and j.is_cuda and i.dtype == torch.int32 and j.dtype == torch.int32
    n = i.numel()
    words = torch.empty((n, 4), dtype=torch.int32, device="cuda")
    _check(lib().mfh_debug_philox(seed, stream_id, i.data_ptr(), j.data_ptr(), n, words.data_ptr(), _stream()))
    return words


def bessel_j_table(x: float, l_max: int):
    """J_l(x), l = 0..l_max, as the library's Chebyshev driver computes them (host only)."""
    import numpy as np
    out = (ctypes.c_double * (l_max + 1))()
    _check(lib().mfh_debug_bessel_j(float(x), int(l_max), out))
    return np.array(out[:])


MIXES = {"c128_pair": 0, "c64_entry": 1, "philox": 2, "dfma31": 3, "comp_philox": 4, "comp_philox_bm_c128": 5,
         "comp_mac_c128": 6, "comp_philox_bm_c64": 7, "comp_mac_c64": 8, "pipe_wide16": 9, "pipe_lop32": 10,
         "pipe_dfma32": 11, "pipe_dfma32_reg3": 12, "pipe_wide16_dfma32": 13, "pipe_lop32_dfma32": 14,
         "pipe_wide16_lop32": 15, "pipe_cmac_regs": 16, "pipe_cmac_lds": 17}


def pipe_rate(mix: str) -> float:
    """Units per second of the synthetic instruction-mix kernel (mfh_debug_pipe_rates)."""
    out = ctypes.c_double(0.0)
    _check(lib().mfh_debug_pipe_rates(MIXES[mix], ctypes.byref(out), _stream()))
    return float(out.value)


def read_bandwidth(buf) -> float:
    """Bytes per second of a read-only stream over a device tensor (mfh_debug_read_bandwidth)."""
    out = ctypes.c_double(0.0)
    _check(lib().mfh_debug_read_bandwidth(buf.data_ptr(), buf.numel() * buf.element_size(), ctypes.byref(out), _stream()))
    return float(out.value)
