"""Delay-depth tuning.

The paper gives only a rule of thumb for the delay depth -- T ~ n/10k for determinants,
T ~ n/20k for Pfaffians -- and says the optimum "depends strongly on the hardware and matrix
size" and that users "perform their own benchmarks".  This
module is that benchmark as a call:

* ``tune_delay(kind, n, k, ...)`` times short chains of the real hot path (propose -> ratio ->
  decide -> accept/flush, the same ``mc.Chain`` bench.py times) at each candidate depth K on
  the current GPU and returns the fastest, with the whole table;
* ``recommended_delay(kind, n, k, dtype)`` answers without measuring: the depth measured on
  B200 for the nearest tuned shape (``tuned_delay_b200.json``, written by
  ``python -m paper_2602_05255_b200.tune --write-table``), else the paper's rule of thumb.

Orchestration only: every timed step runs in the library's kernels; inputs are the seeded
synthetic workload of DESIGN.md §4.
"""
from __future__ import annotations

import argparse
import json
import math
import os

HERE = os.path.dirname(os.path.abspath(__file__))
TABLE_PATH = os.path.join(HERE, "tuned_delay_b200.json")
DEPTHS = (0, 2, 4, 8, 16, 32, 64)


def heuristic_delay(kind, n, k):
    """The paper's rule of thumb: T ~ n/10k (det), n/20k (Pfaffian)."""
    return max(0, int(n // ((10 if kind == "det" else 20) * k)))


def _walkers_for(kind, n, cplx, budget_bytes):
    esz = 16 if cplx else 8
    per = n * n * esz * (2 + (2 if kind == "det" else 4))      # inverse + A0 scratch + orbitals
    return int(max(148, min(16384, budget_bytes // per)))


def tune_delay(kind, n, k, cplx=False, W=None, depths=DEPTHS, steps=None, mode="metropolis", seed=20260205,
               device=None, budget_bytes=3e10):
    """Measure walker-updates/s of the hot path at each delay depth in ``depths`` (0 = immediate
    updates) and return {"best": K, "table": [...], "heuristic": K_paper, ...}.

    ``mode``: "metropolis" (the chain as the configs write it; acceptance 0.15-0.45, so a walker
    fills its buffer every K/acc steps) or "forced" (every proposal applied: the paper's Fig. 2
    setting).  ``steps`` defaults to enough steps for every depth to flush at
    least twice.  Depths the library rejects for this shape (LRUX_EUNSUPPORTED) are skipped.
    """
    import torch

    from . import lrux, mc
    from . import workload as wl

    device = torch.device("cuda", torch.cuda.current_device()) if device is None else device
    M = 2 * n
    W = _walkers_for(kind, n, cplx, budget_bytes) if W is None else int(W)
    if kind == "det":
        orb = wl.orbital_matrices_torch(seed, 0, W, M, n, (0.5 if cplx else 1.0) / n, device, cplx)
    else:
        if cplx:
            raise ValueError("the synthetic Pfaffian workload is real-valued")
        orb = wl.pairing_matrices_torch(seed, 0, W, M, 1.0 / n, device)
    occ, unocc = wl.initial_occupations(seed, W, M, n)
    occ_t, unocc_t = torch.as_tensor(occ, device=device), torch.as_tensor(unocc, device=device)
    forced = mode == "forced"
    acc_guess = 1.0 if forced else 0.25
    table = []
    for K in depths:
        if K > 0 and K * k >= n:
            continue                                  # T < n/k
        try:
            ch = mc.Chain(kind, orb, occ_t.clone(), unocc_t.clone(), k=k, K=K, seed=seed)
        except lrux.LruxError as e:
            if e.status == lrux.EUNSUPPORTED:
                continue
            raise
        warm = int(math.ceil(max(K, 1) / acc_guess)) + 2          # buffers reach their steady state
        nsteps = steps or max(20, int(math.ceil(2 * max(K, 1) / acc_guess)))
        for t in range(warm):
            ch.step(t, forced)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for t in range(nsteps):
            ch.step(warm + t, forced)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / nsteps
        table.append({"K": K, "ms_per_step": ms, "walker_updates_per_s": W / (ms * 1e-3), "steps": nsteps})
        del ch
    best = max(table, key=lambda r: r["walker_updates_per_s"])
    base = next((r for r in table if r["K"] == 0), None)
    return {"kind": kind, "n": n, "k": k, "dtype": "c128" if cplx else "f64", "W": W, "mode": mode,
            "best": best["K"], "speedup_vs_immediate": (best["walker_updates_per_s"] / base["walker_updates_per_s"]
                                                         if base else None),
            "heuristic": heuristic_delay(kind, n, k), "table": table}


_TABLE = None


def load_table():
    global _TABLE
    if _TABLE is None:
        try:
            _TABLE = json.load(open(TABLE_PATH))["entries"]
        except (OSError, ValueError, KeyError):
            _TABLE = []
    return _TABLE


def recommended_delay(kind, n, k, cplx=False):
    """Delay depth for this shape without measuring: the depth tuned on B200 for the nearest
    shape of the same kind / dtype (distance in log2 n and log2 k), else the paper's rule."""
    dt = "c128" if cplx else "f64"
    cand = [e for e in load_table() if e["kind"] == kind and e["dtype"] == dt]
    if not cand:
        return heuristic_delay(kind, n, k)
    d = lambda e: abs(math.log2(e["n"] / n)) + abs(math.log2(e["k"] / k))
    e = min(cand, key=d)
    if d(e) > 1.5:
        return heuristic_delay(kind, n, k)
    K = int(e["best"])
    return K if K * k < n else heuristic_delay(kind, n, k)


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--kind", default="det", choices=["det", "pf"])
    ap.add_argument("--n", type=int, default=512)
    ap.add_argument("--k", type=int, default=1)
    ap.add_argument("--cplx", action="store_true")
    ap.add_argument("--mode", default="metropolis", choices=["metropolis", "forced"])
    ap.add_argument("--walkers", type=int, default=0)
    ap.add_argument("--write-table", action="store_true",
                    help="tune the grid of shapes below and write tuned_delay_b200.json")
    args = ap.parse_args(argv)
    if not args.write_table:
        print(json.dumps(tune_delay(args.kind, args.n, args.k, args.cplx, W=args.walkers or None, mode=args.mode)))
        return 0
    import torch

    entries = []
    grid = [("det", n, k, False) for n in (128, 256, 512, 1024, 2048) for k in (1, 2, 4, 8)]
    grid += [("det", 1024, 4, True)]
    grid += [("pf", n, k, False) for n in (128, 256, 512) for k in (1, 2, 4)]
    for kind, n, k, cplx in grid:
        r = tune_delay(kind, n, k, cplx, mode=args.mode)
        entries.append({key: r[key] for key in ("kind", "n", "k", "dtype", "W", "mode", "best", "speedup_vs_immediate",
                                                "heuristic")}
                       | {"table": [{"K": t["K"], "walker_updates_per_s": round(t["walker_updates_per_s"])}
                                    for t in r["table"]]})
        print(json.dumps(entries[-1]), flush=True)
        torch.cuda.empty_cache()
    json.dump({"gpu": torch.cuda.get_device_name(), "command": "python -m paper_2602_05255_b200.tune --write-table",
               "entries": entries}, open(TABLE_PATH, "w"), indent=1)
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
