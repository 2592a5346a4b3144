#!/usr/bin/env python
"""bench.py -- throughput of the hot path phi = H psi on B200 (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W            # the CUDA path (default N=1)
    python bench.py --impl reference --steps K --warmup W    # the CPU oracle, as it stands

A "step" is one pass of the whole hot path over one batch of synthetic input: one mfh_apply of the
planned Hamiltonian on one normalised random psi.  At N=1 the workload is BASELINE.json
configs[1] ("C2": D=65536, complex128, B=2048, full cache, 68.7 GB resident in HBM), the
configuration the HBM-bound metric is quoted on.  The path does not shard (north_star: one GPU,
no collectives): --gpus N runs N independent replicas ("replicas only") and the value
is the sum over ranks divided by the max-over-ranks time.

Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every field.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2606_31598_b200.inputs import (CONFIGS, SYSTEM_BATH, VARIANTS, lambda_grid, make_psi, sample_rows,  # noqa: E402
                                          small_hermitian)

ALL = dict(CONFIGS, **VARIANTS)

METRIC = "matrix_entries_per_s"
UNIT = "entries/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---- clocks during the timed region (B200_PROFILING.md recipe) --------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---- CPU oracle legs (the only places bench.py may execute oracle/) ---------------------------
def oracle_rows_apply(cfg: dict, psi, rows):
    import oracle
    if cfg["k"] > 1:
        return oracle.apply_scan(cfg["D"], cfg["B"], cfg["seed"], cfg["seed_h0"], lambda_grid(cfg["k"]),
                                 psi, rows=rows)
    return oracle.apply(cfg["D"], cfg["B"], cfg["seed"], psi, rows=rows)


def cpu_info() -> dict:
    model = "unknown"
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count()}


def cpu_baseline(cfg: dict, psi, target_s: float = 15.0) -> dict:
    """The oracle as it stands, timed on the host cores on a bounded row sample of the workload."""
    import oracle
    D = cfg["D"]
    probe = sample_rows(D, 250, seed=1)[:256]
    t0 = time.perf_counter()
    oracle_rows_apply(cfg, psi, probe)
    dt = time.perf_counter() - t0
    n = int(min(max(len(probe) * target_s / max(dt, 1e-6), 256), D))
    rows = np.arange(n, dtype=np.int64) * (D // n)
    t0 = time.perf_counter()
    oracle_rows_apply(cfg, psi, rows)
    dt = time.perf_counter() - t0
    return {"value": n * D / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", **cpu_info(),
            "omp_threads": oracle.num_threads(), "entries_per_s_per_core": n * D / dt / max(oracle.num_threads(), 1),
            "sample": f"{n} evenly spaced output rows of {D} ({n * D:.3g} matrix entries, {dt:.1f} s); "
                      f"implied full apply {D * D / (n * D / dt):.0f} s (extrapolated)"}


def run_reference(args, cfg_name: str):
    """--impl reference: the oracle on the same config/metric; each step a bounded row sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cfg = ALL[cfg_name]
    D = cfg["D"]
    psi = make_psi(D, cfg["psi_seed"], k=cfg["k"], dtype=cfg["dtype"])
    n = max(64, min(D, int(2.0e8 / D)))          # ~2e8 entries per step: a few seconds on 8 cores
    rows = np.arange(n, dtype=np.int64) * (D // n)
    for _ in range(args.warmup):
        oracle_rows_apply(cfg, psi, rows[: max(8, n // 8)])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_rows_apply(cfg, psi, rows)
    dt = time.perf_counter() - t0
    value = args.steps * n * D / dt
    sample = f"{n} evenly spaced output rows of {D} per step ({n * D:.3g} entries)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(cfg_name, cfg),
            "applies_per_s": value / (D * D),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", **cpu_info(),
                             "omp_threads": oracle.num_threads(), "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(name: str, cfg: dict) -> dict:
    return {"workload": f"{name}: seeded GUE D={cfg['D']} {cfg['dtype']} B={cfg['B']} {cfg['mode']} k={cfg['k']}",
            "D": cfg["D"], "B": cfg["B"], "mode": cfg["mode"], "k": cfg["k"],
            "l2_policy": "inputs larger than L2 (cached blocks)" if cfg["mode"] != "procedural"
            else "no L2-resident input: entries are generated in registers; vectors only (flushed between steps)"}


# ---- the CUDA path ---------------------------------------------------------------------------
def make_handle(mfh, cfg: dict, n_applies: int):
    kind = "diag_plus_gue" if "seed_h0" in cfg else "gue"
    h = mfh.Hamiltonian(cfg["D"], cfg["B"], cfg["seed"], cfg["dtype"], kind=kind, seed_h0=cfg.get("seed_h0", 0))
    plan = h.plan(cfg["mode"], k=cfg["k"], n_applies_hint=n_applies,
                  hbm_budget_bytes=int(cfg.get("hbm_budget", 0)))
    return h, plan


def time_steps(torch, fn, steps: int, flush=None):
    """CUDA-event time of `steps` calls on the current stream (ms total).  With `flush`, every step
    has its own event pair and the L2 flush runs between pairs, outside the timed spans."""
    if flush is None:
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(steps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b)
    pairs = []
    for _ in range(steps):
        flush()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        pairs.append((a, b))
    torch.cuda.synchronize()
    return sum(a.elapsed_time(b) for a, b in pairs)


def measure_config(torch, mfh, name: str, steps: int, warmup: int, with_e2e: bool, barrier=None):
    cfg = ALL[name]
    D, k = cfg["D"], cfg["k"]
    psi_np = make_psi(D, cfg["psi_seed"], k=k, dtype=cfg["dtype"])
    lam = lambda_grid(k) if k > 1 else None
    t0 = time.perf_counter()
    # configs[4] (C5) is one Chebyshev propagation of 151 applies: that is the job its plan is made for
    h, plan = make_handle(mfh, cfg, 151 if "t" in cfg else max(steps, 1))
    torch.cuda.synchronize()
    plan_s = time.perf_counter() - t0
    info = h.get_plan()
    psi = torch.from_numpy(psi_np).cuda()
    phi = torch.empty_like(psi)
    flush_buf = None
    flush = None
    if cfg["mode"] == "procedural":
        flush_buf = torch.empty(256 * 2**20, dtype=torch.uint8, device="cuda")   # > 126 MB L2
        flush = lambda: flush_buf.fill_(1)  # noqa: E731
    fn = lambda: h.apply(psi, phi, lambdas=lam)  # noqa: E731
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    # per-kernel durations from the SAME pass: mfh_timing_begin arms event records around each launch of the next
    # K applies (no synchronisation inside the pass), so kernel_ms.total <= ms_per_step by construction
    h.timing_begin(steps)
    ms = time_steps(torch, fn, steps, flush)
    recs = h.timing_end()
    if barrier:
        barrier()
    assert len(recs) == steps, (len(recs), steps)
    kern = {key: sum(r[key] for r in recs) / steps for key in ("cached", "procedural", "reduce", "total")}
    out = {"name": name, "cfg": cfg, "pipe_rate": mfh.pipe_rate, "plan": info, "plan_s": plan_s, "ms_total": ms, "steps": steps,
           "ms_per_step": ms / steps, "kernel_ms": kern, "psi_np": psi_np,
           "launches_per_apply": info["launches_per_apply"]}
    if "t" in cfg and k == 1:
        # BASELINE.json configs[4]: one Chebyshev propagation e^{-iHt} psi (K-1 applies), timed with events
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        outv, K = h.chebyshev(psi, cfg["t"], cfg["e_min"], cfg["e_max"], cfg["tol"])
        b.record()
        torch.cuda.synchronize()
        out["chebyshev"] = {"t": cfg["t"], "tol": cfg["tol"], "bounds": [cfg["e_min"], cfg["e_max"]], "terms": K,
                            "applies": K - 1, "seconds": a.elapsed_time(b) * 1e-3,
                            "norm_error": abs(float(torch.linalg.vector_norm(outv).item()) - 1.0)}
        del outv
        # NEXT-2: the bounds the paper's way, from 40 matrix-free Lanczos steps with a 5 % margin
        t0 = time.perf_counter()
        e0, e1, _, _ = h.lanczos_bounds(psi, m=40, margin=0.05)
        out["chebyshev"]["lanczos_bounds"] = {"m": 40, "margin": 0.05, "e_min": e0, "e_max": e1,
                                              "seconds": time.perf_counter() - t0}
    if with_e2e:
        ph = torch.from_numpy(psi_np).pin_memory()
        oh = torch.empty_like(ph).pin_memory()
        for _ in range(max(1, warmup)):
            h.apply_host(ph, oh, lambdas=lam)
        e_ms = time_steps(torch, lambda: h.apply_host(ph, oh, lambdas=lam), steps)
        out["e2e_ms_per_step"] = e_ms / steps
        out["io_bytes"] = ph.numel() * ph.element_size()
    h.destroy()
    del psi, phi, flush_buf
    torch.cuda.empty_cache()
    return out


def measure_system_bath(torch, mfh, steps: int, hbm_gbs: float, mode: str = None) -> dict:
    """NEXT-3: the paper's own workload shape: 18 qubits, two cached dense complex64
    bath-side operators (32 GiB each) applied to R = d_S = 4 columns; operators synthetic (R19)."""
    c = SYSTEM_BATH
    d_B, d_S = c["d_B"], c["d_S"]
    sb = mfh.SystemBath(d_B, d_S, c["B"], c["seed_HB"], c["seed_B1"], small_hermitian(d_S, c["seed_HS"]),
                        small_hermitian(d_S, c["seed_A"]), c["g"], dtype=c["dtype"])
    t0 = time.perf_counter()
    plan = sb.plan(mode or c["mode"], n_applies_hint=steps)
    torch.cuda.synchronize()
    plan_s = time.perf_counter() - t0
    X = torch.from_numpy(make_psi(d_B, c["psi_seed"], k=d_S, dtype=c["dtype"])).cuda()
    Y = torch.empty_like(X)
    for _ in range(3):
        sb.apply(X, Y)
    torch.cuda.synchronize()
    ms = time_steps(torch, lambda: sb.apply(X, Y), steps) / steps
    nbytes = plan["H_B"]["cache_bytes"] + plan["B_1"]["cache_bytes"]
    sb.destroy()
    del X, Y
    torch.cuda.empty_cache()
    if mode == "pairs":
        nbytes_read = 2 * nbytes - 2 * (d_B // c["B"]) * c["B"] ** 2 * 8     # every off-diagonal stored block is read twice
        return {"workload": f"system-bath 18 qubits from two Hermitian pair caches ({nbytes / 1e9:.1f} GB stored): the mirrored "
                            "positions are served by a second, transposed read of the stored blocks",
                "ms_per_apply": ms, "applies_per_s": 1e3 / ms, "stored_bytes": nbytes, "bytes_read_per_apply": nbytes_read,
                "achieved_gbs": nbytes_read / (ms * 1e-3) / 1e9, "plan_and_fill_s": plan_s}
    return {"workload": f"system-bath 18 qubits: d_S={d_S}, d_B={d_B}, {c['dtype']}, B={c['B']}, 2 cached bath operators x {d_S} columns",
            "ms_per_apply": ms, "applies_per_s": 1e3 / ms, "flops_per_apply": plan["flops_per_apply"],
            "cached_bytes": nbytes, "achieved_gbs": nbytes / (ms * 1e-3) / 1e9, "frac_of_measured_hbm": nbytes / (ms * 1e-3) / 1e9 / hbm_gbs,
            "plan_and_fill_s": plan_s,
            "paper": {"seconds_per_apply": c["paper_seconds_per_apply"], "hardware": c["paper_hardware"],
                      "note": "context only: other machine, the paper's own (unpublished) operators",
                      "ratio_paper_over_this": c["paper_seconds_per_apply"] / (ms * 1e-3)}}


def measure_partition_projection(torch, mfh, name: str = "C4", worlds=(2, 8), steps: int = 3) -> dict:
    """NEXT-4 on one GPU: the local apply time of rank 0 of a W-GPU job (mfh_set_partition), which is what
    every rank of the job would spend between two exchanges of D * B_c bytes.  The exchange itself (NCCL over
    NVSwitch) cannot be timed on this one-GPU box and is NOT included."""
    cfg = ALL[name]
    D = cfg["D"]
    psi = torch.from_numpy(make_psi(D, cfg["psi_seed"], dtype=cfg["dtype"])).cuda()
    phi = torch.zeros_like(psi)
    flush_buf = torch.empty(256 * 2**20, dtype=torch.uint8, device="cuda")
    out = {"workload": workload_config(name, cfg)["workload"], "exchange_bytes_per_apply": psi.numel() * psi.element_size(),
           "note": "per-rank kernel time of rank 0, exchange not included (one-GPU box)", "ranks": {}}
    for scheme in ("rows", "pairs"):
        for W in worlds:
            h = mfh.Hamiltonian(D, cfg["B"], cfg["seed"], cfg["dtype"])
            h.set_partition(0, W, scheme)
            h.plan(cfg["mode"], k=1, hbm_budget_bytes=int(cfg.get("hbm_budget", 0)))
            for _ in range(2):
                h.apply(psi, phi)
            torch.cuda.synchronize()
            ms = time_steps(torch, lambda: h.apply(psi, phi), steps, lambda: flush_buf.fill_(1)) / steps
            out["ranks"][f"{scheme}/W={W}"] = {"ms_per_apply_rank0": ms, "owned_blocks": h.get_plan()["partition"]["owned_blocks"],
                                               "projected_entries_per_s_job": D * D / (ms * 1e-3)}
            h.destroy()
    return out


def measure_graph_replay(torch, mfh, name: str = "C1", n: int = 50) -> dict:
    """Launch-bound regime (C1: 76 us per apply, 3 launches): n applies and one Chebyshev propagation captured in
    CUDA graphs and replayed, against the same calls issued eagerly."""
    cfg = ALL[name]
    D = cfg["D"]
    h, _ = make_handle(mfh, cfg, n)
    psi = torch.from_numpy(make_psi(D, cfg["psi_seed"], dtype=cfg["dtype"])).cuda()
    phi = torch.empty_like(psi)
    out = torch.empty_like(psi)
    for _ in range(3):
        h.apply(psi, phi)
    h.chebyshev(psi, 50.0, -2.1, 2.1, 1e-14, out=out)
    torch.cuda.synchronize()
    eager_ms = time_steps(torch, lambda: h.apply(psi, phi), n) / n
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    _, K = h.chebyshev(psi, 50.0, -2.1, 2.1, 1e-14, out=out)
    b.record()
    torch.cuda.synchronize()
    cheb_eager_ms = a.elapsed_time(b)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g_apply, g_cheb = torch.cuda.CUDAGraph(), torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(g_apply, stream=s):
            for _ in range(n):
                h.apply(psi, phi)
        with torch.cuda.graph(g_cheb, stream=s):
            h.chebyshev(psi, 50.0, -2.1, 2.1, 1e-14, out=out)
    torch.cuda.synchronize()
    g_apply.replay(); g_cheb.replay()
    torch.cuda.synchronize()
    graph_ms = time_steps(torch, g_apply.replay, 3) / (3 * n)
    cheb_graph_ms = time_steps(torch, g_cheb.replay, 3) / 3
    h.destroy()
    return {"workload": workload_config(name, cfg)["workload"], "applies_in_graph": n,
            "ms_per_apply_eager": eager_ms, "ms_per_apply_graph": graph_ms,
            "chebyshev": {"t": 50.0, "terms": K, "ms_eager": cheb_eager_ms, "ms_graph": cheb_graph_ms}}


def measure_auto_planner(torch, mfh) -> dict:
    """a-6 end to end: mfh_plan(AUTO, B = 0, measure = 1) (Algorithm 2: the K_bench <= 8 best analytic candidates timed
    on the device, argmin of n_applies x measured time + fill) on the operators of C2 (100 applies), C5 (151 applies
    inside 150 GB) and C3 (100 scans): which plan it commits, its measured apply time and how long planning took."""
    out = {}
    for name, n_applies in (("C2", 100), ("C5", 151), ("C3", 100)):
        cfg = ALL[name]
        kind = "diag_plus_gue" if "seed_h0" in cfg else "gue"
        h = mfh.Hamiltonian(cfg["D"], 0, cfg["seed"], cfg["dtype"], kind=kind, seed_h0=cfg.get("seed_h0", 0))
        t0 = time.perf_counter()
        rec = h.plan("auto", k=cfg["k"], n_applies_hint=n_applies, hbm_budget_bytes=int(cfg.get("hbm_budget", 0)), measure=True)
        torch.cuda.synchronize()
        c = rec["chosen"]
        out[name] = {"operator": f"D={cfg['D']} {cfg['dtype']} k={cfg['k']}", "n_applies_hint": n_applies,
                     "chosen": {kk: c[kk] for kk in ("mode", "B", "cache_bytes", "cached_fraction")},
                     "measured_ms_per_apply": c["measured_apply_s"] * 1e3, "model_ms_per_apply": c["model_apply_s"] * 1e3,
                     "matrix_entries_per_s": cfg["D"] ** 2 / c["measured_apply_s"],
                     "candidates_timed": sum(1 for x in rec["candidates"] if x["measured_apply_s"] > 0),
                     "plan_seconds": time.perf_counter() - t0}
        h.destroy()
        torch.cuda.empty_cache()
    return out


def measure_pipe_model(mfh) -> dict:
    """Which instruction classes of the generator overlap on this GPU: units/s of the library's
    synthetic kernels and the clocks one warp instruction of the class costs a scheduler at 1.965 GHz nominal.  A pair
    of classes that takes the sum of its parts does not overlap."""
    n = {"pipe_wide16": 32, "pipe_lop32": 32, "pipe_dfma32": 33, "pipe_dfma32_reg3": 33, "pipe_wide16_dfma32": 65,
         "pipe_lop32_dfma32": 65, "pipe_wide16_lop32": 64, "pipe_cmac_regs": 1, "pipe_cmac_lds": 1}
    out = {}
    for name, instr in n.items():
        r = mfh.pipe_rate(name)
        clk = 148 * 4 * 1.965e9 / (r / 32.0)      # scheduler clocks per warp-unit
        out[name] = {"units_per_s": r, "clk_per_warp_unit": clk, "instructions_per_unit": instr}
    c = {k: v["clk_per_warp_unit"] for k, v in out.items()}
    out["summary"] = {
        "dfma_clk_immediate_operands": c["pipe_dfma32"] / 33, "dfma_clk_three_register_operands": c["pipe_dfma32_reg3"] / 33,
        "wide_plus_dfma_over_sum": c["pipe_wide16_dfma32"] / (c["pipe_wide16"] + c["pipe_dfma32"]),
        "lop_plus_dfma_over_max": c["pipe_lop32_dfma32"] / max(c["pipe_lop32"], c["pipe_dfma32"]),
        "wide_plus_lop_over_sum": c["pipe_wide16_lop32"] / (c["pipe_wide16"] + c["pipe_lop32"]),
        "dfma_clk_mac_stream_one_operand_reused": c["pipe_cmac_regs"], "dfma_clk_k_vector_inner_loop": c["pipe_cmac_lds"],
        "fp64_peak_fraction_with_three_register_dfma": (c["pipe_dfma32"] / 33) / (c["pipe_dfma32_reg3"] / 33) * (2.0 / (c["pipe_dfma32"] / 33)),
        "note": "ratios near 1.0 over the SUM mean the two classes serialise (32x32->64 multiply against DFMA and "
                "against logic ops); near 1.0 over the MAX mean they overlap (logic ops under DFMA)"}
    return out


def roofline_for(res: dict, hbm_gbs: float, peak_src: str) -> dict:
    """Roofline of the dominant kernel of one apply."""
    cfg = res["cfg"]
    D, k = cfg["D"], cfg["k"]
    kern = res["kernel_ms"]
    if res["plan"]["mode"] == "partial" and kern["cached"] < 0.01 * kern["procedural"]:
        # overlapped partial mode: ONE kernel streams the cached blocks and generates the rest (Eq. 33);
        # its HBM roofline is the cached bytes over the whole kernel time
        nbytes = res["plan"]["cache_bytes"]
        gbs = nbytes / (kern["procedural"] * 1e-3) / 1e9
        gen = D * D * (1.0 - res["plan"]["cached_fraction"]) / (kern["procedural"] * 1e-3)
        return {"kernel": "partial_overlap_kernel", "bound": "hbm", "achieved": gbs, "peak": hbm_gbs, "unit": "GB/s",
                "frac": gbs / hbm_gbs, **ncu_traffic("partial_overlap_kernel", D), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": nbytes, "kernel_ms": kern["procedural"],
                "generated_entries_per_s_in_the_same_kernel": gen,
                "share_of_step": kern["procedural"] / max(kern["total"], 1e-9)}
    if kern["cached"] >= kern["procedural"] and k >= 8 and cfg["dtype"] == "c128":
        # cached complex128 blocks on k >= 8 vectors: 4k DFMA per 16-byte entry, FP64-pipe bound
        flops = 8.0 * D * D * k * res["plan"]["cached_fraction"]
        tf = flops / (kern["cached"] * 1e-3) / 1e12
        peak = 148 * 64 * 2 * 1.965e9 / 1e12
        # second number: the rate at which DFMAs with three register operands issue on this GPU (measured now); the
        # kernel's multiply-accumulates read the entry, the psi value and the accumulator from registers
        reg3 = res["pipe_rate"]("pipe_dfma32_reg3") * 33 * 2 / 1e12
        # third and fourth number: the complex multiply-accumulate stream alone (psi in registers: all but the first DFMA
        # of a run take the entry from the operand reuse cache, 2 clocks each) and this kernel's inner loop as written
        # (entry and psi values from shared memory every column), both measured now by the library's microbenchmarks
        cmac_regs = res["pipe_rate"]("pipe_cmac_regs") * 2 / 1e12
        cmac_lds = res["pipe_rate"]("pipe_cmac_lds") * 2 / 1e12
        return {"kernel": "cached_multi_kernel_c128", "bound": "alu", "achieved": tf, "peak": peak, "unit": "TFLOP/s",
                "frac": tf / peak, **ncu_traffic("cached_multi_kernel_c128", D),
                "three_register_dfma_ceiling": reg3, "frac_of_three_register_dfma_ceiling": tf / reg3,
                "mac_stream_in_registers_ceiling": cmac_regs, "inner_loop_from_shared_memory_ceiling": cmac_lds,
                "frac_of_inner_loop_ceiling": tf / cmac_lds,
                "peak_source": "nominal FP64: 148 SMs x 64 DFMA lanes/clk x 2 flop x 1.965 GHz (B200_PROFILING.md unit counts; "
                               "the SM clock under FP64 load is power-capped below that)",
                "kernel_ms": kern["cached"], "share_of_step": kern["cached"] / max(kern["total"], 1e-9)}
    if kern["cached"] >= kern["procedural"]:
        # HBM-bound cached streaming: algorithmic bytes = stored entries * bytes per entry
        nbytes = res["plan"]["cache_bytes"]
        one_read = res["plan"].get("two_sided_stored_pairs", 0) > 0   # unit-image layout: both positions from one read
        if res["plan"]["mode"] == "pairs" and k > 1 and not one_read:
            # k-vector pair cache without the unit-image layout: every stored off-diagonal block is read twice
            nb = D // cfg["B"]
            nbytes = 2 * nbytes - nb * cfg["B"] ** 2 * (8 if cfg["dtype"] == "c64" else 16)
        gbs = nbytes / (kern["cached"] * 1e-3) / 1e9
        name = "cached_pairs_kernel" if (res["plan"]["mode"] == "pairs" and k == 1) else (
            "cached_kernel" if k == 1 else (("pairs_tc_kernel<true>" if one_read else "cached_multi_tc_kernel") if cfg["dtype"] == "c64" else "cached_multi_kernel_c128"))
        out = {"kernel": name, "bound": "hbm", "achieved": gbs, "peak": hbm_gbs, "unit": "GB/s",
               "frac": gbs / hbm_gbs, **ncu_traffic(name, cfg["D"]), "peak_source": peak_src,
               "algorithmic_bytes_per_launch": nbytes, "kernel_ms": kern["cached"],
               "share_of_step": kern["cached"] / max(kern["total"], 1e-9)}
        if one_read:
            # half the bytes of the full cache for the same entries: the HBM fraction halves by construction; what
            # bounds this kernel is on-chip (ncu: tensor pipe 72 %, shared memory 74 %, SM clock power-capped to 1.5 GHz)
            nb = D // cfg["B"]
            out["applied_bytes_equivalent_gbs"] = (2 * nbytes - nb * cfg["B"] ** 2 * 8) / (kern["cached"] * 1e-3) / 1e9
            out["note"] = ("every stored block is read once and serves both positions; bound by the tensor pipe and shared "
                           "memory (profiles/r02_pairs_tc_cached_c3_ncu_full.md), not by HBM")
        return out
    # ALU-bound fused generate-and-apply: unit = matrix entries applied per second by that kernel.
    # Headline denominator = an implementation-independent pipe peak from the guide's unit counts and clocks: the FP64
    # pipe for the complex128 kernel (64 DFMA lanes/clk/SM), the issue slots for the complex64 tensor-core generator;
    # the measured instruction-mix ceiling and the component ceilings (the library's own generator functions, one
    # component at a time) are reported beside it.
    entries = D * D * (1.0 - res["plan"]["cached_fraction"])
    rate = entries / (kern["procedural"] * 1e-3)
    key = (cfg["dtype"], "k1" if k == 1 else "kN")
    two_sided = k > 1 and res["plan"].get("two_sided_pairs", 0) > 0   # block pairs generated once for both positions
    if two_sided:
        key = (cfg["dtype"], "kN2")
    cnt = SASS_COUNTS[key]
    issue_peak = ISSUE_LANES_PER_S / cnt["instr_per_entry"]
    kname = "proc_single_kernel" if k == 1 else (("pairs_tc_kernel<false>" if two_sided else "proc_multi_tc_kernel") if cfg["dtype"] == "c64" else "proc_multi_kernel")
    out = {"kernel": kname, "bound": "alu", "achieved": rate / 1e9, "unit": "Gentries/s", **ncu_traffic(kname, D),
           "issue_slot_peak": issue_peak / 1e9, "frac_of_issue_slots": rate / issue_peak,
           "instr_per_entry": cnt["instr_per_entry"], "sass_counts_source": cnt["source"],
           "kernel_ms": kern["procedural"], "share_of_step": kern["procedural"] / max(kern["total"], 1e-9)}
    if cnt.get("fp64_per_entry"):
        fp64_peak = FP64_LANES_PER_S / cnt["fp64_per_entry"]
        out.update({"peak": fp64_peak / 1e9, "frac": rate / fp64_peak, "fp64_per_entry": cnt["fp64_per_entry"],
                    "peak_source": f"FP64 pipe: 148 SMs x 64 DFMA lanes/clk x 1.965 GHz (B200_PROFILING.md unit counts and clocks) / "
                                   f"{cnt['fp64_per_entry']} FP64 instructions per entry in the inner loop's SASS ({cnt['source']}); "
                                   "nominal clock, the run itself is power-capped below it (see clocks)"})
    else:
        out.update({"peak": issue_peak / 1e9, "frac": rate / issue_peak,
                    "peak_source": f"issue slots: 148 SMs x 4 warp instructions/clk x 1.965 GHz / {cnt['instr_per_entry']} instructions "
                                   f"per entry in the inner loop's SASS ({cnt['source']})"})
    mix = MIX_OF.get(key)
    if mix is not None:
        # second number: ceiling measured live on this GPU by a synthetic kernel with the inner loop's instruction counts
        name, entries_per_unit = mix
        if two_sided:   # applied entries per generated entry: both positions of a pair from one generation
            nb = D // cfg["B"]
            entries_per_unit = nb * nb / (nb * nb - res["plan"]["two_sided_pairs"])
        mix_peak = res["pipe_rate"](name) * entries_per_unit
        out.update({"mix_ceiling": mix_peak / 1e9, "frac_of_mix_ceiling": rate / mix_peak,
                    "mix_ceiling_source": f"measured now: mfh_debug_pipe_rates({name}) x {entries_per_unit} entries per unit "
                                          "(synthetic kernel with the per-entry IMAD.WIDE/LOP3/DFMA/MUFU/FFMA counts, DESIGN.md 6.2)"})
    comp = COMPONENTS_OF.get(key)
    if comp is not None:
        # Philox-only, Philox+Box-Muller and MAC-only micro-kernels built from the library's own device
        # functions; generated pairs/s, two entries per pair with Hermitian reuse, one entry per pair without
        epp = comp["entries_per_pair"]
        r = {nm: res["pipe_rate"](nm) * epp for nm in comp["kernels"]}
        gen, mac = r[comp["kernels"][1]], r[comp["kernels"][2]]
        serial = 1.0 / (1.0 / gen + 1.0 / mac)
        out["components"] = {"unit": "Gentries/s", "philox_only": r[comp["kernels"][0]] / 1e9, "philox_box_muller": gen / 1e9,
                             "mac_only": mac / 1e9, "harmonic_gen_plus_mac": serial / 1e9,
                             "frac_of_harmonic": rate / serial, "frac_of_generation_alone": rate / gen}
    return out


# ALU ceilings.  Instruction counts per matrix entry come from the SASS of the inner loops (cuobjdump;
# tables in profiles/).  Nominal pipe peaks: every SM issues at most 4 warp instructions per clock and has 64 FP64
# lanes (B200_PROFILING.md unit counts, 1.965 GHz).
ISSUE_LANES_PER_S = 148 * 4 * 32 * 1.965e9
FP64_LANES_PER_S = 148 * 64 * 1.965e9
SASS_COUNTS = {("c128", "k1"): {"instr_per_entry": 43.875, "fp64_per_entry": 16.0, "source": "profiles/r02_proc_single_sass.md"},
               ("c128", "kN"): {"instr_per_entry": 150.0, "fp64_per_entry": 0, "source": "DESIGN.md 6.3"},
               ("c64", "k1"): {"instr_per_entry": 40.0, "fp64_per_entry": 0, "source": "DESIGN.md 6.2"},
               ("c64", "kN"): {"instr_per_entry": 64.0, "fp64_per_entry": 0, "source": "profiles/r02_proc_multi_tc_c3_ncu_full.md (2.14e9 warp instructions / 1.07e9 entries x 32 lanes)"},
               # two-sided generator: everything the step executes, per APPLIED entry (generator 63.5 per generated entry
               # in its SASS; epilogue, sum, MMA warps and barrier waits on top; the one-sided kernel for the diagonal blocks)
               ("c64", "kN2"): {"instr_per_entry": 38.3, "fp64_per_entry": 0,
                                "source": "profiles/r02_pairs_tc_generated_c3_ncu_full.md + r02_proc_multi_tc_diag_c3_ncu_full.md "
                                          "((1.217e9 + 0.069e9) warp instructions / 1.07e9 applied entries x 32 lanes)"}}
MIX_OF = {("c128", "k1"): ("c128_pair", 2), ("c64", "kN"): ("c64_entry", 1), ("c64", "kN2"): ("c64_entry", 1)}
COMPONENTS_OF = {("c128", "k1"): {"kernels": ("comp_philox", "comp_philox_bm_c128", "comp_mac_c128"), "entries_per_pair": 2},
                 ("c64", "k1"): {"kernels": ("comp_philox", "comp_philox_bm_c64", "comp_mac_c64"), "entries_per_pair": 2}}


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full captures, keyed by
# (kernel, D): (bytes per launch, the capture it was read from).  A kernel without a capture reports "traffic": null.
NCU_TRAFFIC = {("cached_kernel", 65536): (68.725132e9 + 5.106432e6, "profiles/r02_cached_c2_ncu_full.md"),
               ("partial_overlap_kernel", 131072): (146.236774e9 + 252.962816e6, "profiles/r02_partial_overlap_c5_ncu_full.md"),
               ("cached_pairs_kernel", 65536): (35.438780e9 + 249.902592e6, "profiles/r01_pairs_c2_ncu_full.md"),
               ("cached_multi_tc_kernel", 32768): (8.595266e9 + 135.4e6, "profiles/r02_cached_multi_tc_c3_ncu_full.md"),
               ("cached_multi_kernel_c128", 32768): (17.203616e9 + 268.850432e6, "profiles/r02_cached_multi_c128_c3_ncu_full.md"),
               ("proc_single_kernel", 262144): (22.890752e6 + 631.663104e6, "profiles/r02_proc_single_c4_ncu_full.md"),
               ("proc_multi_tc_kernel", 32768): (4.513792e6 + 81.728768e6, "profiles/r02_proc_multi_tc_c3_ncu_full.md"),
               ("pairs_tc_kernel<false>", 32768): (6.530304e6 + 527.058688e6, "profiles/r02_pairs_tc_generated_c3_ncu_full.md"),
               ("pairs_tc_kernel<true>", 32768): (4.219875e9 + 583.816448e6, "profiles/r02_pairs_tc_cached_c3_ncu_full.md")}


def ncu_traffic(kernel: str, D: int) -> dict:
    """Traffic of a committed ncu capture (not measured in this run: bench.py never runs under a profiler) and the
    file it came from."""
    v = NCU_TRAFFIC.get((kernel, D))
    return {"traffic": v[0] if v else None, "traffic_source": v[1] if v else None}


def add_read_probe(rf: dict, read_probe_gbs):
    """Beside the contract's frac (against the driver-measured COPY peak): the fraction of a read-only stream
    measured in this run by the library's probe kernel, the fairer ceiling for a kernel that only reads."""
    if rf.get("bound") == "hbm" and read_probe_gbs:
        rf["read_only_probe_gbs"] = read_probe_gbs
        rf["frac_of_read_only_probe"] = rf["achieved"] / read_probe_gbs
    return rf


def aggregate(dist, local_ms: float, local_units: float, device=None):
    """max-over-ranks time and sum-over-ranks units (works with nccl and gloo)."""
    if dist is None:
        return local_ms, local_units
    import torch
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def run_partitioned(torch, dist, args, rank: int, world: int, local: int):
    """--partition rows|pairs with N > 1 (NEXT-4): one operator over the N GPUs, every step = local apply +
    one NCCL exchange of D * B_c bytes; value = D^2 entries per step over the max-over-ranks time."""
    from paper_2606_31598_b200.distributed import DistributedHamiltonian
    cfg = ALL[args.workload]
    D, k = cfg["D"], cfg["k"]
    kind = "diag_plus_gue" if "seed_h0" in cfg else "gue"
    dh = DistributedHamiltonian(D, cfg["B"], cfg["seed"], cfg["dtype"], kind=kind, seed_h0=cfg.get("seed_h0", 0),
                                scheme=args.partition)
    dh.plan(mode=cfg["mode"], k=k, n_applies_hint=args.steps, hbm_budget_bytes=int(cfg.get("hbm_budget", 0)))
    info = dh.h.get_plan()
    psi = torch.from_numpy(make_psi(D, cfg["psi_seed"], k=k, dtype=cfg["dtype"])).cuda()
    phi = torch.zeros_like(psi)
    lam = lambda_grid(k) if k > 1 else None
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(args.warmup):
        dh.apply(psi, phi, lam)
    torch.cuda.synchronize()
    dist.barrier()
    torch.cuda.synchronize()
    ms_local = time_steps(torch, lambda: dh.apply(psi, phi, lam), args.steps)
    dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop() if rank == 0 else None
    ms, _ = aggregate(dist, ms_local, 0.0, torch.device("cuda", local))
    value = args.steps * float(D) * D / (ms * 1e-3)
    if rank == 0:
        wc = workload_config(args.workload, cfg)
        wc["partition"] = {"scheme": args.partition, "world": world, "exchange_bytes_per_apply": psi.numel() * psi.element_size()}
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                          "scaling": "strong", "vs_baseline": None, "dtype": "f64" if cfg["dtype"] == "c128" else "f32",
                          "data": "synthetic", "config": wc, "applies_per_s": value / (float(D) * D), "plan": info,
                          "gpu_launches": info["launches_per_apply"] * args.steps, "clocks": clocks,
                          "e2e": None, "roofline": None, "cpu_baseline": None}), flush=True)
    dh.destroy()
    dist.barrier()
    dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="C2", choices=sorted(ALL))
    ap.add_argument("--partition", default="none", choices=["none", "rows", "pairs"],
                    help="N > 1 only: ONE operator over the N GPUs (mfh_set_partition + one NCCL exchange per apply, "
                         "strong scaling) instead of N replicas")
    ap.add_argument("--no-extra", action="store_true", help="skip the other configs' side measurements")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--save", default="", help="also write the JSON line (with other_configs) to this file")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup

    if args.impl == "reference":
        run_reference(args, args.workload)
        return

    import torch
    from paper_2606_31598_b200 import binding as mfh
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    mfh.lib()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    barrier = (lambda: (dist.barrier(), torch.cuda.synchronize())) if dist else None

    if args.partition != "none":
        if dist is None:   # one GPU: a single-rank group, so that the same code path runs (and is tested) here
            import torch.distributed as dist
            import socket
            with socket.socket() as sk:   # any free port: nothing else joins this group
                sk.bind(("127.0.0.1", 0))
                port = sk.getsockname()[1]
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", str(port))
            dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", local))
        run_partitioned(torch, dist, args, rank, world, local)
        return

    hbm_gbs, peak_src = load_peaks()
    read_probe_gbs = None
    if rank == 0:
        # read-only stream probe: the copy peak of MEASURED_PEAKS.json pays a write turn-around that a
        # kernel reading a cached matrix once does not; 16 GiB, far above L2
        probe = torch.empty(16 * 2**30, dtype=torch.uint8, device="cuda")
        probe.fill_(1)
        read_probe_gbs = mfh.read_bandwidth(probe) / 1e9
        del probe
        torch.cuda.empty_cache()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    res = measure_config(torch, mfh, args.workload, args.steps, args.warmup, with_e2e=True, barrier=barrier)
    clocks = sampler.stop() if rank == 0 else None

    cfg = res["cfg"]
    D = cfg["D"]
    dev = torch.device("cuda", local)
    ms, units = aggregate(dist, res["ms_total"], float(args.steps) * D * D, dev)
    e_ms, _ = aggregate(dist, res["e2e_ms_per_step"] * args.steps, 0.0, dev)
    value = units / (ms * 1e-3)
    e2e_value = units / (e_ms * 1e-3)

    extras = {}
    if rank == 0 and world == 1 and not args.no_extra:
        for name, st in (("C1", 20), ("C3", 5), ("C3-cached", 10), ("C3-pairs", 10), ("C3-c128-cached", 5), ("C4", 3), ("C2-pairs", 10),
                         ("C5", 3), ("C5-pairs", 5)):
            if name == args.workload:
                continue
            try:
                r = measure_config(torch, mfh, name, st, 3, with_e2e=False)
                rf = add_read_probe(roofline_for(r, hbm_gbs, peak_src), read_probe_gbs)
                c = r["cfg"]
                extras[name] = {"workload": workload_config(name, c)["workload"], "steps": st,
                                "plan": {kk: r["plan"][kk] for kk in ("mode", "B", "cached_fraction", "cache_bytes")},
                                "ms_per_apply": r["ms_per_step"], "applies_per_s": 1e3 / r["ms_per_step"],
                                "matrix_entries_per_s": c["D"] ** 2 / (r["ms_per_step"] * 1e-3),
                                "kernel_ms": r["kernel_ms"], "roofline": rf, "plan_s": r["plan_s"]}
                if "chebyshev" in r:
                    extras[name]["chebyshev"] = r["chebyshev"]
            except Exception as e:  # a side measurement must not lose the headline line
                extras[name] = {"error": str(e)}
        try:
            extras["SB18"] = measure_system_bath(torch, mfh, 10, hbm_gbs)
        except Exception as e:
            extras["SB18"] = {"error": str(e)}
        try:
            extras["SB18-pairs"] = measure_system_bath(torch, mfh, 10, hbm_gbs, mode="pairs")
        except Exception as e:
            extras["SB18-pairs"] = {"error": str(e)}
        try:
            extras["planner-auto-measured"] = measure_auto_planner(torch, mfh)
        except Exception as e:
            extras["planner-auto-measured"] = {"error": str(e)}
        try:
            extras["C1-graph"] = measure_graph_replay(torch, mfh)
        except Exception as e:
            extras["C1-graph"] = {"error": str(e)}
        try:
            extras["pipe-model"] = measure_pipe_model(mfh)
        except Exception as e:
            extras["pipe-model"] = {"error": str(e)}
        try:
            extras["C4-partitioned"] = measure_partition_projection(torch, mfh)
        except Exception as e:
            extras["C4-partitioned"] = {"error": str(e)}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64" if cfg["dtype"] == "c128" else "f32",
                "data": "synthetic", "config": workload_config(args.workload, cfg),
                "applies_per_s": value / (D * D), "plan": res["plan"], "plan_and_fill_s": res["plan_s"],
                "kernel_ms": res["kernel_ms"], "roofline": add_read_probe(roofline_for(res, hbm_gbs, peak_src), read_probe_gbs),
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": res["io_bytes"],
                        "d2h_bytes_per_step": res["io_bytes"], "ms_per_step": e_ms / args.steps},
                "gpu_launches": res["launches_per_apply"] * args.steps, "clocks": clocks,
                "other_configs": extras}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(cfg, res["psi_np"])
        else:
            line["cpu_baseline"] = None
        print(json.dumps(line), flush=True)
        if args.save:
            os.makedirs(os.path.dirname(os.path.abspath(args.save)), exist_ok=True)
            with open(args.save, "w") as f:
                json.dump(line, f, indent=1)
                f.write("\n")
    if dist:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
