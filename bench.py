#!/usr/bin/env python
"""bench.py -- walker-updates/s of the lrux hot path on B200 (BASELINE.json metric).

One "step" = one Monte-Carlo step of every walker through the whole hot path
(SURVEY.md §8(a)): lruxh_*_propose -> lrux_*_ratio -> lruxh_decide -> lrux_*_accept
(immediate Woodbury update, or delayed append + flush when K > 0), all enqueued on
one CUDA stream without host synchronisation.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c4|n512...]
    python bench.py --impl reference        # the CPU oracle on the host cores

Prints ONE JSON line (rank 0).  See DESIGN.md §7 for the definition of every key.
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

METRIC = "walker_updates_per_s"
UNIT = "walker-updates/s"

# name -> kind, dtype, W (per GPU), n, M, k, K variants (first = headline), default steps
WORKLOADS = {
    # BASELINE.json configs[1]: the configuration the metric is quoted on
    "c2": dict(kind="det", cplx=False, W=4096, n=256, M=512, k=2, Ks=(0, 16), cfg=2,
               desc="configs[1]: det f64, 4096 walkers, n=256, M=512, k=2, Metropolis; K=0 vs K=16"),
    "c3": dict(kind="pf", cplx=False, W=1024, n=128, M=256, k=1, Ks=(0, 4), cfg=3,
               desc="configs[2]: pf f64, 1024 walkers, n=128, M=256, k=1, Metropolis"),
    "c4": dict(kind="det", cplx=True, W=512, n=1024, M=2048, k=4, Ks=(32,), cfg=4,
               desc="configs[3]: det c128, 512 walkers, n=1024, M=2048, k=4, K=32, Metropolis"),
    # small case used by the tests of bench.py itself
    "tiny": dict(kind="det", cplx=False, W=64, n=64, M=128, k=2, Ks=(0, 4), cfg=2,
                 desc="tiny det f64 smoke workload"),
}


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="lrux", choices=["lrux", "reference"])
    ap.add_argument("--workload", default="c2")
    ap.add_argument("--walkers", type=int, default=0, help="override walkers per GPU")
    ap.add_argument("--e2e-steps", type=int, default=16)
    ap.add_argument("--cpu-seconds", type=float, default=15.0,
                    help="CPU time budget of the cpu_baseline sample")
    ap.add_argument("--mode", default="metropolis", choices=["metropolis", "forced"],
                    help="forced: every proposal is applied (ncu captures, Fig. 2-style runs)")
    ap.add_argument("--delay", type=int, default=-1,
                    help="override the workload's delay depth K (headline variant only)")
    ap.add_argument("--no-graph", action="store_true",
                    help="time stream-launched steps instead of CUDA-graph replays")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip forced-accept / delayed variants / DGEMM yardstick")
    return ap.parse_args(argv)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        """Launch nvidia-smi and wait (<= 3 s) for its first sample, so that the sampler
        is already running when the timed region begins."""
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
            t0 = time.perf_counter()
            while not self.lines and time.perf_counter() - t0 < 3.0:
                time.sleep(0.01)
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def mark_begin(self):
        self.t_begin = time.perf_counter()

    def stop(self):
        t_end = time.perf_counter()
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.03)          # let a sample that straddles the end arrive
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        t_begin = getattr(self, "t_begin", 0.0)
        inside = [ln for (t, ln) in self.lines if t_begin <= t <= t_end + 0.03]
        if not inside:            # timed region shorter than one sampling period: nearest samples
            inside = [ln for (_, ln) in self.lines[-2:]]
        sm, smax, reasons, power = [], [], set(), []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in inside:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None,
                "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------- GPU arm
def build_inputs(wk, W, w0, device):
    """Seeded synthetic inputs of the workload's shape, generated on the device
    (DESIGN.md §4): per-walker Phi (det) or skew F (pf) and the initial occupation."""
    from paper_2602_05255_b200 import workload as wl

    seed = wl.BASE_SEED + wk["cfg"]
    n, M = wk["n"], wk["M"]
    if wk["kind"] == "det":
        var = 1.0 / (2 * n) if wk["cplx"] else 1.0 / n
        orb = wl.orbital_matrices_torch(seed, w0, W, M, n, var, device, wk["cplx"])
    else:
        orb = wl.pairing_matrices_torch(seed, w0, W, M, 1.0 / n, device)
    occ, unocc = wl.initial_occupations(seed, W, M, n, w0=w0)
    return seed, orb, occ, unocc


_MASTERS = {}     # K -> (pristine initialised walkers, init seconds): init runs once per K
INIT_SECONDS = {}


def make_chain(wk, K, seed, orb, occ, unocc, w0, device):
    """A chain at step 0.  The O(n^3) initialisation (step a0, timed separately and
    reported as init_s) runs once per delay depth; every chain then starts from a byte
    copy of that state (lrux_*_attach)."""
    import torch
    from paper_2602_05255_b200 import mc

    occ_t, unocc_t = torch.as_tensor(occ, device=device), torch.as_tensor(unocc, device=device)
    if K not in _MASTERS:
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        first = mc.Chain(wk["kind"], orb, occ_t, unocc_t, k=wk["k"], K=K, seed=seed, w0=w0)
        torch.cuda.synchronize()
        INIT_SECONDS[K] = time.perf_counter() - t0      # includes the gather of A0 from the orbitals
        _MASTERS[K] = first.walkers
    return mc.Chain(wk["kind"], orb, occ_t, unocc_t, k=wk["k"], K=K, seed=seed, w0=w0,
                    walkers=_MASTERS[K].clone())


def timed_run(ch, warmup, steps, forced=False, sampler=None, graph=True):
    """W untimed + K timed steps; device time by CUDA events on the launching stream,
    barrier + synchronize on both sides.  ``graph``: the timed steps are K replays of ONE
    step captured into a CUDA graph (the step counter lives in device memory: mc.Chain.capture);
    the warm-up steps and the profiled pass are plain stream launches of the same sequence.
    A second pass of K more steps, stream-launched with the library's per-class CUDA events
    switched on, gives the per-kernel durations the roofline figures use (events between
    the launches of a replayed graph would only keep their last recording).
    Returns a dict of raw measurements."""
    import torch
    from paper_2602_05255_b200 import lrux, shard

    for t in range(warmup):
        ch.step(t, forced)
    torch.cuda.synchronize()
    launch = "stream"
    if graph:
        try:
            ch.capture(warmup, forced)
            launch = "cuda_graph"
        except Exception as e:        # capture refused: fall back to stream launches, say so
            launch = "stream (graph capture failed: %s)" % type(e).__name__
    torch.cuda.synchronize()
    shard.barrier()
    torch.cuda.synchronize()
    acc0 = int(ch.naccept.item())
    l0 = ch.launches()
    if sampler:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if sampler:
        sampler.mark_begin()
        torch.cuda.profiler.start()   # ncu --profile-from-start off sees the timed region only
    e0.record()
    if launch == "cuda_graph":
        for t in range(steps):
            ch.replay()
    else:
        for t in range(steps):
            ch.step(warmup + t, forced)
    e1.record()
    torch.cuda.synchronize()
    if sampler:
        torch.cuda.profiler.stop()
    shard.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    ms = e0.elapsed_time(e1)
    accepted = int(ch.naccept.item()) - acc0
    launches = steps * ch.launches_per_replay if launch == "cuda_graph" else ch.launches() - l0

    # ---- profiled pass: the next `steps` steps of the same chain, per-class events on
    acc1 = int(ch.naccept.item())
    f0 = ch.walkers.flush_count() if ch.K > 0 else (0, 0)
    ch.walkers.profile_enable(True)
    for c in range(5):
        ch.walkers.profile_read(c)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    for t in range(steps):
        ch.step(warmup + steps + t, forced)
    p1.record()
    torch.cuda.synchronize()
    prof = {}
    for name, c in (("ratio", lrux.PROF_RATIO), ("update", lrux.PROF_UPDATE),
                    ("append", lrux.PROF_APPEND), ("flush", lrux.PROF_FLUSH),
                    ("ypass", lrux.PROF_YPASS)):
        t_ms, cnt = ch.walkers.profile_read(c)
        prof[name] = {"ms": t_ms, "launches": cnt}
    ch.walkers.profile_enable(False)
    f1 = ch.walkers.flush_count() if ch.K > 0 else (0, 0)
    kernels = {name: ch.walkers.kernel_name(c) for name, c in
               (("ratio", lrux.PROF_RATIO), ("update", lrux.PROF_UPDATE), ("append", lrux.PROF_APPEND),
                ("flush", lrux.PROF_FLUSH), ("ypass", lrux.PROF_YPASS))}
    return {"ms": ms, "accepted_timed": accepted, "launches": launches, "launch": launch,
            # the profiled pass: what the per-kernel roofline figures are computed from
            "accepted": int(ch.naccept.item()) - acc1, "ms_profiled_pass": p0.elapsed_time(p1),
            "flushes": f1[0] - f0[0], "flush_cols": f1[1] - f0[1],
            "prof": prof, "clocks": clocks, "kernels": kernels}


def e2e_run(wk, seed, orb, occ, unocc, w0, device, warmup, steps):
    """The same chain driven through the C-ABI calls from HOST buffers: every step
    copies idx + new rows from pinned host memory, reads the ratios back, takes the
    Metropolis decision on the host and uploads the mask.  The host
    inputs are recorded from a device-harness run of the same chain beforehand, so
    the replay walks the identical trajectory."""
    import numpy as np
    import torch
    from paper_2602_05255_b200 import workload as wl

    K = wk["Ks"][0]
    T = warmup + steps
    W, k, n = occ.shape[0], wk["k"], wk["n"]
    dt = orb.dtype
    rec = make_chain(wk, K, seed, orb, occ, unocc, w0, device)
    # bring the chain to its steady state first (delay buffers in every stage of filling)
    # with the device harness, then snapshot it: the replay starts from that snapshot
    pre = 3 * K
    for t in range(pre):
        rec.step(t)
    torch.cuda.synchronize()
    from paper_2602_05255_b200 import mc
    A0_chain = mc.Chain(wk["kind"], orb, rec.occ.clone(), rec.unocc.clone(), k=k, K=K, seed=seed,
                        w0=w0, walkers=rec.walkers.clone())
    idx_h = torch.empty((T, W, k), dtype=torch.int32).pin_memory()
    rows_h = torch.empty((T, W, k, n), dtype=dt).pin_memory()
    mask_rec = torch.empty((T, W), dtype=torch.uint8).pin_memory()
    for t in range(T):
        rec.step(pre + t)
        idx_h[t].copy_(rec.idx)
        rows_h[t].copy_(rec.rows)
        mask_rec[t].copy_(rec.mask)
    torch.cuda.synchronize()
    wkr = A0_chain.walkers
    del rec
    xi = np.stack([wl.to_uniform(wl.rnd64(seed, np.arange(w0, w0 + W, dtype=np.uint64),
                                          wl.STREAM_ACCEPT, np.uint64(pre + t))) for t in range(T)])
    mask_d = A0_chain.mask
    # two sets of device input buffers: the upload of step t+1 (copy stream) overlaps the
    # host decision and the accept of step t (compute stream)
    idx_d = [A0_chain.idx, torch.empty_like(A0_chain.idx)]
    rows_d = [A0_chain.rows, torch.empty_like(A0_chain.rows)]
    ratio_h = torch.empty(W, dtype=dt).pin_memory()
    mask_h = torch.empty(W, dtype=torch.uint8).pin_memory()
    main = torch.cuda.current_stream()
    cs = torch.cuda.Stream()
    copied = [torch.cuda.Event(), torch.cuda.Event()]

    def upload(t):
        b = t & 1
        with torch.cuda.stream(cs):
            idx_d[b].copy_(idx_h[t], non_blocking=True)
            rows_d[b].copy_(rows_h[t], non_blocking=True)
            copied[b].record(cs)

    mism = 0
    t_start = 0.0
    upload(0)
    for t in range(T):
        if t == warmup:
            torch.cuda.synchronize()
            t_start = time.perf_counter()
        b = t & 1
        main.wait_event(copied[b])
        wkr.ratio_(idx_d[b], rows_d[b])           # copies what accept needs into the state
        ratio_h.copy_(wkr.ratio, non_blocking=True)
        if t + 1 < T:
            upload(t + 1)                         # buffer 1-b: its ratio finished last step
        main.synchronize()
        r = ratio_h.numpy()
        a2 = r.real ** 2 + r.imag ** 2 if wk["cplx"] else r * r
        m = (xi[t] < np.minimum(1.0, a2))
        mask_h.numpy()[:] = m
        mism += int((m != mask_rec[t].numpy().astype(bool)).sum())
        mask_d.copy_(mask_h, non_blocking=True)
        wkr.accept(mask_d)
    torch.cuda.synchronize()
    sec = time.perf_counter() - t_start
    esz = 16 if wk["cplx"] else 8
    return {"sec": sec, "steps": steps, "mismatch": mism,
            "h2d": W * k * 4 + W * k * n * esz + W, "d2h": W * esz}


# ---------------------------------------------------------------------------- CPU oracle arm
def oracle_sample(wk, warmup, steps, budget_s, walkers=0):
    """Time the oracle AS IT STANDS (oracle/lrux_oracle_c.c: plain loops, no BLAS, gcc -O2) on
    the host cores: walkers 0..Wc-1 of the workload (Wc = 4 x cores unless given), one OpenMP
    thread per walker in flight, all cores busy, the oracle's naive path only (lemma ratio +
    Eq. 5 / Eq. 21 Woodbury update or the delayed carrier; no from-scratch recomputation:
    scratch_every = 0).  Each walker clocks its own steps >= `warmup` (the O(n^3)
    initialisation and the warm-up steps are left out); throughput = walker-steps /
    (sum of those times / threads), i.e. what the box sustains with every core on a walker.
    A short probe sizes T <= `steps` so that the timed part stays near `budget_s` seconds.
    Returns (seconds, walker-steps, walkers, threads, T)."""
    import numpy as np
    from oracle import c_oracle
    from paper_2602_05255_b200 import workload as wl

    seed = wl.BASE_SEED + wk["cfg"]
    n, M, k, K = wk["n"], wk["M"], wk["k"], wk["Ks"][0]
    threads = c_oracle.num_threads()
    Wc = walkers or min(wk["W"], 4 * threads)
    used = min(threads, Wc)
    if wk["kind"] == "det":
        var = 1.0 / (2 * n) if wk["cplx"] else 1.0 / n
        orb = np.stack([wl.orbital_matrix(seed, w, M, n, var, wk["cplx"]) for w in range(Wc)])
    else:
        orb = np.stack([wl.pairing_matrix(seed, w, M, 1.0 / n, wk["cplx"]) for w in range(Wc)])
    occ, unocc = wl.initial_occupations(seed, Wc, M, n)

    def run(nw, T):
        P, J, xi = wl.proposals(seed, nw, warmup + T, n, M, k)
        res = c_oracle.batch(wk["kind"], orb[:nw], occ[:nw], unocc[:nw], P, J, xi, scratch_every=0, delay=K,
                             final_scratch=False, want_matrices=False, mark_step=warmup)
        return sum(r["seconds"] for r in res) / min(used, nw)

    probe = max(1, min(steps, 4))
    per_step = max(run(used, probe) / probe, 1e-7) * Wc / used       # one step of all Wc walkers
    T = int(max(1, min(steps, budget_s / per_step)))
    sec = max(run(Wc, T), 1e-9)
    return sec, Wc * T, Wc, used, T


def reference_arm(args, wk):
    """--impl reference: the oracle timed on the host cores on this arm's config,
    metric and unit (rank 0 only)."""
    from paper_2602_05255_b200 import shard

    rank, _, _ = shard.env_rank()
    if rank != 0:
        return 0
    steps, warmup = args.steps, args.warmup
    # each step of this arm is a bounded sample of the workload's step: Wc walkers instead of W
    sec, done, nw, cores, T = oracle_sample(wk, warmup, steps, args.cpu_seconds * 2)
    value = done / sec
    sample = ("%d of %d walkers x %d steps of %s (after %d warm-up steps), C oracle naive path, "
              "one OpenMP thread per walker in flight" % (nw, wk["W"], T, args.workload, max(1, warmup)))
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
           "n_gpus": args.gpus, "steps": steps, "warmup": warmup,
           "ms_per_step": 1e3 * sec / max(1, T), "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "c128" if wk["cplx"] else "f64", "data": "synthetic",
           "config": {"workload": wk["desc"], "K": wk["Ks"][0], "sample": sample},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))
    return 0


# ---------------------------------------------------------------------------- main
def dgemm_yardstick(device, n=4096, reps=5):
    """cuBLAS FP64 GEMM throughput (TFLOP/s) as the measured FP64 tensor peak the
    flush is reported against (yardstick only; not on the product path)."""
    import torch

    a = torch.randn((n, n), dtype=torch.float64, device=device)
    b = torch.randn((n, n), dtype=torch.float64, device=device)
    torch.matmul(a, b)
    torch.cuda.synchronize()
    best = 1e30
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        torch.matmul(a, b)
        e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    return 2.0 * n ** 3 / (best * 1e-3) / 1e12


def ncu_traffic_per_walker(kernel, workload):
    """(DRAM bytes per updated walker, source file) from the newest committed `ncu --set full`
    capture of this kernel on this workload (profiles/*_traffic.csv); (None, None) when there
    is none.  NOT measured in the bench run: the bench line says where it comes from."""
    import csv
    import glob

    best = (None, None)
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "*_traffic.csv"))):
        for row in csv.DictReader(open(path)):
            if row["kernel"] == kernel and row["workload"] == workload:
                best = ((float(row["dram_bytes_read"]) + float(row["dram_bytes_write"]))
                        / float(row["walkers_updated_per_launch"]), os.path.relpath(path, ROOT))
    return best


def roofline_update(wk, run, peak, peak_src, dgemm_tflops=None):
    """HBM roofline of the immediate Woodbury update kernel:
    algorithmic bytes = 2 n^2 e per accepted walker (read once + write once).  Ranks k > 8
     are above the FP64 ridge (k/4 flop/B): reported against the FP64 tensor
    roofline, algorithmic flops = 4 n^2 k per accepted walker (u^T A^-1 and the rank-k apply)."""
    esz = 16 if wk["cplx"] else 8
    pr = run["prof"]["update"]
    if pr["launches"] == 0 or pr["ms"] <= 0:
        return None
    byts = 2.0 * wk["n"] ** 2 * esz * run["accepted"]
    ach = byts / (pr["ms"] * 1e-3) / 1e9
    kern = run.get("kernels", {}).get("update", "")      # as reported by the library (lrux_kernel_name)
    if wk["k"] > 8 and dgemm_tflops:
        tf = 4.0 * wk["n"] ** 2 * wk["k"] * (4 if wk["cplx"] else 1) * run["accepted"] / (pr["ms"] * 1e-3) / 1e12
        return {"bound": "tensor", "kernel": kern, "achieved": tf, "peak": dgemm_tflops, "unit": "TFLOP/s",
                "frac": tf / dgemm_tflops, "traffic": None, "hbm_gbs_2n2e": ach,
                "peak_source": "cuBLAS FP64 GEMM 4096^3 measured in this run (burst)",
                "us_per_launch": 1e3 * pr["ms"] / pr["launches"], "launches": pr["launches"]}
    tpw, src = ncu_traffic_per_walker(kern, wk.get("name", ""))
    traffic = tpw * run["accepted"] / pr["launches"] if tpw else None
    return {"bound": "hbm", "kernel": kern, "achieved": ach, "peak": peak,
            "unit": "GB/s", "frac": ach / peak, "traffic": traffic,
            "traffic_source": ("committed ncu --set full capture %s, scaled to this run's accepted walkers per "
                               "launch; not measured in this run" % src) if tpw else None,
            "peak_source": peak_src,
            "bytes_per_launch": byts / pr["launches"], "us_per_launch": 1e3 * pr["ms"] / pr["launches"],
            "launches": pr["launches"]}


def roofline_flush(wk, K, run, hbm_peak, hbm_src, dgemm_tflops):
    """Roofline of the flush kernel (a7).  Per accepted update (one of the K slots of a
    flushed buffer): 2 n^2 k flops (x4 complex) and (2 n^2 e)/K + 2 n k e bytes.  Arithmetic
    intensity Kk/8 flop/B (real), Kk/4 (complex): FP64-tensor-bound when Kk >= 50 (real) /
    25 (complex), HBM-bound below.  The tensor peak is the cuBLAS FP64
    GEMM measured in this same run (MEASURED_PEAKS.json carries no FP64 figure)."""
    fl = run["prof"]["flush"]
    if K <= 0 or fl["ms"] <= 0 or run.get("flush_cols", 0) <= 0:
        return None
    cx = wk["cplx"]
    esz = 16 if cx else 8
    n, k = wk["n"], wk["k"]
    pf = wk["kind"] == "pf"
    # exact counts from the library (lrux_get_flush_count): buffer columns folded and walker
    # flushes inside the timed region.  det: 2 n^2 flops per column (x4 complex); pf: the upper
    # triangle only, n^2 per column.  Bytes: 2 n^2 e per flushed walker + 2 n e per column.
    cols, nfl = run["flush_cols"], run["flushes"]
    flops = (1.0 if pf else 2.0) * n * n * cols * (4 if cx else 1)
    byts = 2.0 * n * n * esz * nfl + 2.0 * n * esz * cols
    tf = flops / (fl["ms"] * 1e-3) / 1e12
    gbs = byts / (fl["ms"] * 1e-3) / 1e9
    k = (2 * k) if pf else k      # inner dimension per update
    tensor = K * k >= (25 if cx else 50)
    out = {"kernel": run.get("kernels", {}).get("flush", ""), "Kk": K * k, "tflops": tf, "gbs": gbs,
           "launches": fl["launches"], "ms": fl["ms"]}
    if tensor and dgemm_tflops:
        out.update(bound="tensor", achieved=tf, peak=dgemm_tflops, unit="TFLOP/s",
                   frac=tf / dgemm_tflops, traffic=None,
                   peak_source="cuBLAS FP64 GEMM 4096^3 measured in this run (burst)")
    else:
        out.update(bound="hbm", achieved=gbs, peak=hbm_peak, unit="GB/s", frac=gbs / hbm_peak,
                   traffic=None, peak_source=hbm_src)
    return out


def roofline_append(wk, run, peak, peak_src):
    """HBM roofline of the delayed append class (a6): one read-only pass over A0^-1 = n^2 e
    bytes per accepted walker (det: prep + append kernels; pf, k = 1: the Y pass + append)."""
    if run["prof"]["append"]["ms"] <= 0 or (wk["kind"] == "pf" and wk["k"] > 1):
        return None
    ap_ms = run["prof"]["append"]["ms"] + (run["prof"]["ypass"]["ms"] if wk["kind"] == "pf" else 0.0)
    gbs = wk["n"] ** 2 * (16.0 if wk["cplx"] else 8.0) * run["accepted"] / (ap_ms * 1e-3) / 1e9
    kern = run.get("kernels", {}).get("append", "")
    if wk["kind"] == "pf":
        kern = run.get("kernels", {}).get("ypass", "") + "+" + kern
    return {"bound": "hbm", "kernel": kern, "achieved": gbs, "peak": peak, "unit": "GB/s",
            "frac": gbs / peak, "traffic": None, "peak_source": peak_src, "ms": ap_ms}


def c4_leg(device, peak, peak_src, dgemm, rank, w0_of):
    """The second half of BASELINE.json's metric -- "% FP64 TC peak (flush)" -- needs a
    configuration whose flush is in the tensor regime: configs[3] (complex128, n = 1024,
    k = 4, K = 32: K k = 128).  A short leg of it runs inside the default bench so that the
    driver's record carries it: 160 untimed steps bring the delay buffers to their steady
    state (a walker folds after 32 accepted updates, acceptance ~0.2), then 50 timed steps."""
    import torch

    wk = parse_workload("c4")
    K = wk["Ks"][0]
    seed, orb, occ, unocc = build_inputs(wk, wk["W"], w0_of(wk["W"]), device)
    saved, saved_init = dict(_MASTERS), dict(INIT_SECONDS)
    _MASTERS.clear()
    ch = make_chain(wk, K, seed, orb, occ, unocc, w0_of(wk["W"]), device)
    init_s = INIT_SECONDS.get(K)
    _MASTERS.clear()
    _MASTERS.update(saved)
    INIT_SECONDS.clear()
    INIT_SECONDS.update(saved_init)
    steps, warm = 50, 160
    run = timed_run(ch, warm, steps)
    bad = int((ch.walkers.info != 0).sum().item())
    del ch, orb
    torch.cuda.empty_cache()
    return {"workload": wk["desc"], "steps": steps, "warmup": warm, "init_s": init_s,
            "walker_updates_per_s": wk["W"] * steps / (run["ms"] * 1e-3), "ms_per_step": run["ms"] / steps,
            "accept_frac": run["accepted_timed"] / float(wk["W"] * steps), "info_nonzero_walkers": bad,
            "launch": run["launch"],
            "gpu_launches": run["launches"], "flushes": run["flushes"], "flush_cols": run["flush_cols"],
            "prof_ms": {k: v["ms"] for k, v in run["prof"].items()},
            "roofline_flush": roofline_flush(wk, K, run, peak, peak_src, dgemm),
            "roofline_append": roofline_append(wk, run, peak, peak_src)}


def parse_workload(name):
    """Named workload, or a point of the configs[4] sweep written as
    `det,n=1024,k=4,K=8[,W=2048][,cplx]` / `pf,n=512,k=1,K=0`.  Without W the walker
    count is sized so that inverses + orbital matrices + init scratch fit ~100 GB
    (configs[4] sizes W for 120 GB of inverses alone)."""
    if name in WORKLOADS:
        return dict(WORKLOADS[name], name=name)
    parts = name.split(",")
    if parts[0] not in ("det", "pf"):
        raise SystemExit("unknown workload %r" % name)
    kv = dict(p.split("=") for p in parts[1:] if "=" in p)
    cplx = "cplx" in parts
    n, k, K = int(kv["n"]), int(kv.get("k", 1)), int(kv.get("K", 0))
    esz = 16 if cplx else 8
    # per walker: inverse n^2 + A0 scratch n^2 + orbitals (det: 2 n^2, pf: 4 n^2) + buffers
    per = n * n * esz * (2 + (2 if parts[0] == "det" else 4)) + 2 * K * k * (1 if parts[0] == "det" else 2) * n * esz
    W = int(kv["W"]) if "W" in kv else max(1, int(100e9 // per))
    return dict(kind=parts[0], cplx=cplx, W=W, n=n, M=2 * n, k=k, Ks=(K,), cfg=5, name=name,
                desc="configs[4] sweep point: %s %s, n=%d, M=%d, k=%d, K=%d, %d walkers, Metropolis"
                     % (parts[0], "c128" if cplx else "f64", n, 2 * n, k, K, W))


def main(argv=None):
    args = parse_args(argv)
    wk = parse_workload(args.workload)
    if args.walkers:
        wk["W"] = args.walkers
    if args.delay >= 0:
        wk["Ks"] = (args.delay,)
    if args.impl == "reference":
        return reference_arm(args, wk)

    import torch
    import torch.distributed as dist
    from paper_2602_05255_b200 import build, lrux, shard

    rank, local_rank, world = shard.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    build.build()
    lrux.load_library()

    W = wk["W"]
    w0, _ = shard.walker_range(rank, world, W)
    seed, orb, occ, unocc = build_inputs(wk, W, w0, device)
    peak, peak_src = measured_peaks()
    steps, warmup = args.steps, max(3, args.warmup)

    # headline: first K variant, Metropolis as the config is written
    K0 = wk["Ks"][0]
    ch = make_chain(wk, K0, seed, orb, occ, unocc, w0, device)
    run = timed_run(ch, warmup, steps, forced=args.mode == "forced",
                    sampler=ClockSampler(local_rank) if rank == 0 else None, graph=not args.no_graph)
    info_bad = int((ch.walkers.info != 0).sum().item())
    del ch
    ms_max, = shard.reduce_scalars([run["ms"]], "max", device)
    acc_sum, launches = shard.reduce_scalars([run["accepted_timed"], run["launches"]], "sum", device)
    value = W * world * steps / (ms_max * 1e-3)

    extras = {}
    dgemm = dgemm_yardstick(device) if (rank == 0 and (K0 > 0 or wk["k"] > 8 or not args.no_extras)) else None
    if dgemm:
        extras["dgemm_f64_tflops_cublas"] = dgemm
    if not args.no_extras:
        # forced-accept (every proposal applied: what the paper's Fig. 2 times) -> cleanest roofline
        chf = make_chain(wk, K0, seed, orb, occ, unocc, w0, device)
        fsteps = min(steps, 50)
        rf = timed_run(chf, warmup, fsteps, forced=True)
        del chf
        extras["forced_accept"] = {
            "K": K0, "steps": fsteps, "walker_updates_per_s": W * fsteps / (rf["ms"] * 1e-3),
            "accept_frac": rf["accepted_timed"] / float(W * fsteps),
            "roofline": roofline_update(wk, rf, peak, peak_src, dgemm) if K0 == 0 else None,
            "prof_ms": {k: v["ms"] for k, v in rf["prof"].items()}}
        for K in wk["Ks"][1:]:
            chk = make_chain(wk, K, seed, orb, occ, unocc, w0, device)
            rk = timed_run(chk, warmup, steps)
            del chk
            extras["K%d" % K] = {
                "walker_updates_per_s": W * steps / (rk["ms"] * 1e-3), "ms_per_step": rk["ms"] / steps,
                "accept_frac": rk["accepted_timed"] / float(W * steps),
                "prof_ms": {k: v["ms"] for k, v in rk["prof"].items()},
                "roofline_flush": roofline_flush(wk, K, rk, peak, peak_src, dgemm)}

    # end to end through the C-ABI from host buffers
    e2e_steps = min(args.e2e_steps, steps)
    if e2e_steps > 0:
        ee = e2e_run(wk, seed, orb, occ, unocc, w0, device, 3, e2e_steps)
        ee_sec, = shard.reduce_scalars([ee["sec"]], "max", device)
        e2e_value = W * world * e2e_steps / ee_sec
    else:       # sweep runs (--e2e-steps 0): device-timed figures only
        ee, e2e_value = {"h2d": None, "d2h": None, "mismatch": None}, None

    roof = roofline_update(wk, run, peak, peak_src, dgemm) if K0 == 0 else None
    if roof is None and "forced_accept" in extras and extras["forced_accept"]["roofline"]:
        roof = extras["forced_accept"]["roofline"]
    roof_append = roofline_append(wk, run, peak, peak_src) if K0 > 0 else None
    if roof is None and roof_append is not None:   # the dominant kernel of a delayed configuration
        roof = roof_append
    roof_flush = roofline_flush(wk, K0, run, peak, peak_src, dgemm)

    # the metric's flush half: a short configs[3] leg whenever the headline workload's own flush
    # is not in the FP64-tensor regime (single GPU; the default run)
    if (not args.no_extras and rank == 0 and world == 1 and wk.get("name") != "c4"
            and not (roof_flush and roof_flush.get("bound") == "tensor")):
        del orb
        _MASTERS.clear()
        torch.cuda.empty_cache()
        extras["c4"] = c4_leg(device, peak, peak_src, dgemm, rank, lambda Wc: 0)
        if roof_flush is None and extras["c4"]["roofline_flush"]:
            roof_flush = dict(extras["c4"]["roofline_flush"], workload="configs[3] leg (extras.c4)")
        if roof_append is None and extras["c4"]["roofline_append"]:
            roof_append = dict(extras["c4"]["roofline_append"], workload="configs[3] leg (extras.c4)")

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
           "warmup": warmup, "ms_per_step": ms_max / steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "c128" if wk["cplx"] else "f64",
           "data": "synthetic",
           "config": {"workload": wk["desc"], "walkers_per_gpu": W, "n": wk["n"], "M": wk["M"],
                      "k": wk["k"], "K": K0, "mode": args.mode, "launch": run["launch"],
                      "roofline_region": "second pass of the same number of steps, stream-launched, with the "
                                         "library's per-class CUDA events (prof_ms, ms_profiled_pass)",
                      "l2": "inputs larger than L2: %.2f GiB of inverses per GPU, no flush needed"
                            % (W * wk["n"] ** 2 * (16 if wk["cplx"] else 8) / 2 ** 30)},
           "init_s": {("K%d" % K): v for K, v in INIT_SECONDS.items()},
           "accept_frac": acc_sum / float(W * world * steps),
           "accepted_updates_per_s": acc_sum / (ms_max * 1e-3),
           "gpu_launches": int(launches), "info_nonzero_walkers": info_bad,
           "clocks": run["clocks"],
           "prof_ms": {k: v["ms"] for k, v in run["prof"].items()},
           "ms_profiled_pass": run["ms_profiled_pass"],
           "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": ee["h2d"],
                   "d2h_bytes_per_step": ee["d2h"], "steps": e2e_steps,
                   "decision_mismatches_vs_device_chain": ee["mismatch"]},
           "roofline": roof, "roofline_append": roof_append, "roofline_flush": roof_flush,
           "kernels": run["kernels"], "extras": extras}
    if rank == 0:
        if world == 1 and args.cpu_seconds > 0:
            sec, done, nw, cores, T = oracle_sample(wk, 2, 200, args.cpu_seconds)
            out["cpu_baseline"] = {
                "value": done / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
                "sample": "%d of %d walkers x %d steps of %s (after 2 warm-up steps), C oracle (plain loops, "
                          "no BLAS, gcc -O2) naive path, one OpenMP thread per walker in flight"
                          % (nw, W, T, args.workload)}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
