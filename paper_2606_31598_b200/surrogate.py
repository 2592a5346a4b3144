"""Neural surrogate of the planner (Algorithm 3): marshalling around the library's
``mfh_surrogate_*`` host functions plus the feature vector x(p) of a plan record.

The arithmetic (normalisation, Eq. 24-26, Adam) runs in ``lib/libmfh.so``; this module only builds feature rows from
the JSON records that ``mfh_plan`` / ``mfh_plan_analytic`` return and keeps a portable benchmark log."""
from __future__ import annotations

import ctypes
import json
import math

import numpy as np

from .binding import MFH_OK, MfhError, lib

# x(p) of P:370: (log D, log R, log N_blk, log b, log N_task, p_row, W(p), 1_full, 1_partial, 1_procedural,
# 1_pairs [this build's fourth storage mode], log F_mv, M_op/M_free, M_work/M_free, M_tot/M_free, 1_complex64,
# log GPU memory, log multiprocessors)
FEATURES = ("log_D", "log_R", "log_n_blk", "log_b", "log_n_task", "p_row", "waves", "is_full", "is_partial",
            "is_procedural", "is_pairs", "log_flops", "op_over_free", "work_over_free", "tot_over_free", "is_c64",
            "log_gpu_bytes", "log_sms")
F = len(FEATURES)


def features(D: int, dtype: str, k: int, cand: dict, free_bytes: float, n_task: int = 1, p_row: int = 1, waves: int = 1,
             gpu_bytes: float = 180e9, sms: int = 148) -> np.ndarray:
    """Feature row x(p) of one candidate record (the dicts in plan["candidates"]): marshalling around
    mfh_surrogate_features, which holds the feature map."""
    from .binding import DTYPES, MODES
    out = np.empty(F, dtype=np.float64)
    L = lib()
    L.mfh_surrogate_features.argtypes = [ctypes.c_int64, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32, ctypes.c_int32,
                                         ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int64,
                                         ctypes.c_int32, ctypes.c_int64, ctypes.c_double, ctypes.c_int32,
                                         ctypes.POINTER(ctypes.c_double)]
    rc = L.mfh_surrogate_features(D, DTYPES[dtype], k, MODES[cand["mode"]], int(cand["B"]), float(cand["flops_per_apply"]),
                                  float(cand["cache_bytes"]), float(cand["work_bytes"]), float(free_bytes), int(n_task), int(p_row),
                                  int(waves), float(gpu_bytes), int(sms), _p(out))
    if rc != MFH_OK:
        raise MfhError(rc, lib().mfh_last_error().decode())
    return out


def _p(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _setup():
    L = lib()
    dp, i32, i64 = ctypes.POINTER(ctypes.c_double), ctypes.c_int32, ctypes.c_int64
    L.mfh_surrogate_theta_size.argtypes = [i32, i32]
    L.mfh_surrogate_theta_size.restype = i64
    L.mfh_surrogate_fit.argtypes = [dp, dp, i64, i32, i32, i32, ctypes.c_double, ctypes.c_uint64, dp, dp]
    L.mfh_surrogate_predict.argtypes = [dp, i32, i32, dp, i64, dp]
    L.mfh_surrogate_loss_grad.argtypes = [dp, i32, i32, dp, dp, i64, dp, dp]
    return L


def theta_size(n_features: int, hidden: int) -> int:
    return int(_setup().mfh_surrogate_theta_size(n_features, hidden))


def fit(X, t_seconds, hidden: int = 16, epochs: int = 3000, lr: float = 0.01, seed: int = 0):
    """Train f_theta on records (x_i, t_i); returns (theta, final Eq.-26 loss)."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    t = np.ascontiguousarray(t_seconds, dtype=np.float64)
    n, nf = X.shape
    theta = np.zeros(theta_size(nf, hidden), dtype=np.float64)
    loss = ctypes.c_double(0.0)
    rc = _setup().mfh_surrogate_fit(_p(X), _p(t), n, nf, hidden, epochs, lr, seed, _p(theta), ctypes.byref(loss))
    if rc != MFH_OK:
        raise MfhError(rc, lib().mfh_last_error().decode())
    return theta, float(loss.value)


def predict(theta, X, hidden: int = 16) -> np.ndarray:
    X = np.ascontiguousarray(X, dtype=np.float64).reshape(-1, np.shape(X)[-1])
    out = np.empty(X.shape[0], dtype=np.float64)
    th = np.ascontiguousarray(theta, dtype=np.float64)
    rc = _setup().mfh_surrogate_predict(_p(th), X.shape[1], hidden, _p(X), X.shape[0], _p(out))
    if rc != MFH_OK:
        raise MfhError(rc, lib().mfh_last_error().decode())
    return out


def loss_grad(theta, X, t_seconds, hidden: int = 16):
    X = np.ascontiguousarray(X, dtype=np.float64)
    t = np.ascontiguousarray(t_seconds, dtype=np.float64)
    th = np.ascontiguousarray(theta, dtype=np.float64)
    nf = X.shape[1]
    grad = np.empty(nf * hidden + 2 * hidden + 1, dtype=np.float64)
    loss = ctypes.c_double(0.0)
    rc = _setup().mfh_surrogate_loss_grad(_p(th), nf, hidden, _p(X), _p(t), X.shape[0], ctypes.byref(loss), _p(grad))
    if rc != MFH_OK:
        raise MfhError(rc, lib().mfh_last_error().decode())
    return float(loss.value), grad


def records_from_plan(D: int, dtype: str, k: int, plan: dict, free_bytes: float):
    """(feature row, measured seconds) for every candidate the measured planner timed."""
    out = []
    for c in plan["candidates"]:
        if c.get("measured_apply_s", -1) > 0:
            out.append((features(D, dtype, k, c, free_bytes), c["measured_apply_s"]))
    return out


def rank(theta, D: int, dtype: str, k: int, plan: dict, free_bytes: float, hidden: int = 16):
    """Feasible candidates of an analytic plan record ordered by t_NN(p) W(p) (W = 1 on one GPU)."""
    cands = [c for c in plan["candidates"] if c["feasible"]]
    X = np.stack([features(D, dtype, k, c, free_bytes) for c in cands])
    t = predict(theta, X, hidden)
    order = np.argsort(t)
    return [(cands[i], float(t[i])) for i in order]


def save_log(path: str, rows):
    """Portable benchmark log: one JSON object per line {"x": [...], "t": seconds, "meta": {...}}."""
    with open(path, "w") as f:
        for x, t, meta in rows:
            f.write(json.dumps({"x": [float(v) for v in x], "t": float(t), "meta": meta}) + "\n")


def load_log(path: str):
    X, t, meta = [], [], []
    for line in open(path):
        if line.strip():
            r = json.loads(line)
            X.append(r["x"]); t.append(r["t"]); meta.append(r.get("meta", {}))
    return np.array(X, dtype=np.float64), np.array(t, dtype=np.float64), meta


def hybrid_plan(theta, D: int, dtype: str, k: int = 1, seed: int = 0, kind: str = "gue", seed_h0: int = 0,
                n_applies_hint: int = 1, hbm_budget_bytes: int = 0, k_nn: int = 3, hidden: int = 16, B: int = 0):
    """Algorithm 3, hybrid mode through mfh_plan_hybrid: the library enumerates the memory-feasible candidates,
    ranks them by t_NN(p), commits and times only the top `k_nn` on the device (releasing each before the next) and keeps
    the best measured one (Eq. 23).  Returns (handle with the chosen plan committed, report).  Needs CUDA."""
    from .binding import Hamiltonian, _check, _stream
    h = Hamiltonian(D, B, seed, dtype, kind=kind, seed_h0=seed_h0)
    try:
        th = np.ascontiguousarray(theta, dtype=np.float64)
        assert th.size == theta_size(F, hidden), (th.size, theta_size(F, hidden))
        buf = ctypes.create_string_buffer(1 << 16)
        L = lib()
        L.mfh_plan_hybrid.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.c_int32, ctypes.c_int32, ctypes.c_int64,
                                      ctypes.c_int64, ctypes.c_int32, ctypes.c_void_p, ctypes.c_char_p, ctypes.c_size_t]
        _check(L.mfh_plan_hybrid(h._h, _p(th), hidden, k, n_applies_hint, int(hbm_budget_bytes), k_nn, _stream(), buf, len(buf)))
        h.k = k
        rec = json.loads(buf.value.decode())
    except Exception:
        h.destroy()
        raise
    n = max(n_applies_hint, 1)
    timed = [{"mode": c["mode"], "B": c["B"], "t_nn_s": c["surrogate_apply_s"], "measured_apply_s": c["measured_apply_s"],
              "job_s": n * c["measured_apply_s"] + c["model_fill_s"]} for c in rec["candidates"] if c["measured_apply_s"] > 0]
    c = rec["chosen"]
    chosen = {"mode": c["mode"], "B": c["B"], "t_nn_s": c["surrogate_apply_s"], "measured_apply_s": c["measured_apply_s"],
              "job_s": n * c["measured_apply_s"] + c["model_fill_s"]}
    return h, {"planner": rec["planner"], "feasible_candidates": sum(x["feasible"] for x in rec["candidates"]), "timed": timed,
               "chosen": chosen}
