"""Collect a benchmark log for the planner's neural surrogate (Algorithm 3) on the GPU this runs on,
train the surrogate on part of it and report how well it ranks the held-out problems.

    python -m paper_2606_31598_b200.collect_plan_log --out plan_log.jsonl

Every record is one candidate plan the measured planner (Algorithm 2, mfh_plan with measure = 1) timed:
features x(p) (surrogate.features) and the measured seconds per apply."""
from __future__ import annotations

import argparse
import json

import numpy as np


def collect(problems, budget=0):
    import torch
    from . import binding as mfh
    from . import surrogate as sur
    rows = []
    for (D, dtype, k, n_applies) in problems:
        kind = "diag_plus_gue" if k > 1 else "gue"
        h = mfh.Hamiltonian(D, 0, 1234, dtype, kind=kind, seed_h0=7)
        free = torch.cuda.mem_get_info()[0]
        rec = h.plan("auto", k=k, n_applies_hint=n_applies, hbm_budget_bytes=budget, measure=True)
        for x, t in sur.records_from_plan(D, dtype, k, rec, rec["budget_bytes"]):
            rows.append((x, t, {"D": D, "dtype": dtype, "k": k, "n_applies": n_applies, "free": free}))
        h.destroy()
        torch.cuda.empty_cache()
    return rows


def evaluate(rows, held_out_D, hidden=16, epochs=4000):
    """Train on the problems whose D is not held out; on the held-out ones report the log-time error and the regret
    of the surrogate's first choice (its measured time over the best measured time of that problem)."""
    from . import surrogate as sur
    tr = [r for r in rows if r[2]["D"] not in held_out_D]
    te = [r for r in rows if r[2]["D"] in held_out_D]
    theta, loss = sur.fit(np.stack([r[0] for r in tr]), np.array([r[1] for r in tr]), hidden=hidden, epochs=epochs, lr=0.01, seed=1)
    out = {"train_records": len(tr), "test_records": len(te), "train_loss": loss, "problems": []}
    if te:
        pred = sur.predict(theta, np.stack([r[0] for r in te]), hidden)
        t = np.array([r[1] for r in te])
        out["test_rms_log_error"] = float(np.sqrt(np.mean(np.log(pred / t) ** 2)))
        keys = sorted({(r[2]["D"], r[2]["dtype"], r[2]["k"], r[2]["n_applies"]) for r in te})
        for key in keys:
            idx = [i for i, r in enumerate(te) if (r[2]["D"], r[2]["dtype"], r[2]["k"], r[2]["n_applies"]) == key]
            best = min(t[i] for i in idx)
            pick = idx[int(np.argmin([pred[i] for i in idx]))]
            out["problems"].append({"problem": key, "candidates": len(idx), "best_measured_ms": best * 1e3,
                                    "surrogate_choice_ms": float(t[pick]) * 1e3, "regret": float(t[pick] / best)})
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="plan_log.jsonl")
    ap.add_argument("--report", default="")
    args = ap.parse_args()
    from . import surrogate as sur
    problems = []
    for D in (4096, 8192, 16384, 32768, 65536):
        for dtype in ("c128", "c64"):
            for k, n in ((1, 1), (1, 100), (16, 100)):
                problems.append((D, dtype, k, n))
    rows = collect(problems)
    sur.save_log(args.out, rows)
    rep = evaluate(rows, held_out_D={16384})
    rep["records"] = len(rows)
    print(json.dumps(rep))
    if args.report:
        json.dump(rep, open(args.report, "w"), indent=1)


if __name__ == "__main__":
    main()
