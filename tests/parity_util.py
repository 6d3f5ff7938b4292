"""Helpers for the GPU-vs-oracle parity tests (tests only)."""
import json
import os

import numpy as np
import torch

from oracle import c_oracle as orc          # the compiled restatement (same pins as the numpy one)
from paper_2602_05255_b200 import mc
from paper_2602_05255_b200 import workload as wl

RTOL = 1e-10   # BASELINE.json north_star: relative 1e-10 on ratios and log-amplitudes
CAP = 1e-8     # no point may ever be off by more than this, whatever the conditioning slack
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def make_inputs(kind, seed, W, n, M, cplx=False):
    """Host-generated inputs (identical bytes go to the GPU and to the oracle)."""
    if kind == "det":
        var = 1.0 / (2 * n) if cplx else 1.0 / n
        orb = np.stack([wl.orbital_matrix(seed, w, M, n, var, cplx) for w in range(W)])
    else:
        orb = np.stack([wl.pairing_matrix(seed, w, M, 1.0 / n, cplx) for w in range(W)])
    occ, unocc = wl.initial_occupations(seed, W, M, n)
    return orb, occ, unocc


def current_matrices(ch):
    """A_w of every walker from the chain's occupation (device gather; refresh input)."""
    ar = torch.arange(ch.W, device=ch.orb.device)[:, None]
    occl = ch.occ.long()
    if ch.kind == "det":
        return ch.orb[ar, occl].contiguous()
    return ch.orb[ar[:, :, None], occl[:, :, None], occl[:, None, :]].contiguous()


def record_chain(ch, steps, forced=False, refresh_every=0, sample=None):
    """Run ``steps`` steps of an existing chain, recording ratio, mask and draws of every
    step.  ``forced``: every proposal applied.  ``refresh_every``: lrux_*_refresh from the
    current matrices after every that many steps (the accuracy guard).
    ``sample``: keep the final inverse of these walkers only (full-size runs)."""
    W, k = ch.W, ch.k
    ph0, la0 = ch.walkers.get_amplitude()
    dt = ch.ratio.cpu().numpy().dtype
    rec = dict(ratio=np.zeros((steps, W), dt), mask=np.zeros((steps, W), bool),
               idx=np.zeros((steps, W, k), np.int32), upos=np.zeros((steps, W, k), np.int32),
               init_phase=ph0.cpu().numpy(), init_logabs=la0.cpu().numpy())
    ratio_d = torch.empty((steps, W), dtype=ch.ratio.dtype, device=ch.ratio.device)
    mask_d = torch.empty((steps, W), dtype=torch.uint8, device=ch.ratio.device)
    idx_d = torch.empty((steps, W, k), dtype=torch.int32, device=ch.ratio.device)
    upos_d = torch.empty_like(idx_d)
    for t in range(steps):
        ch.step(t, forced)
        ratio_d[t].copy_(ch.ratio)
        mask_d[t].copy_(ch.mask)
        idx_d[t].copy_(ch.idx)
        upos_d[t].copy_(ch.upos)
        if refresh_every and (t + 1) % refresh_every == 0:
            ch.walkers.refresh(current_matrices(ch))
    rec["ratio"][:] = ratio_d.cpu().numpy()
    rec["mask"][:] = mask_d.cpu().numpy().astype(bool)
    rec["idx"][:] = idx_d.cpu().numpy()
    rec["upos"][:] = upos_d.cpu().numpy()
    ph, la = ch.walkers.get_amplitude()
    full = ch.walkers.get_inverse()
    if sample is None:
        Ainv = full.cpu().numpy()
    else:
        Ainv = _Sparse({w: full[w].cpu().numpy() for w in sample})
    del full
    rec.update(phase=ph.cpu().numpy(), logabs=la.cpu().numpy(), Ainv=Ainv, occ=ch.occ.cpu().numpy(),
               unocc=ch.unocc.cpu().numpy(), info=ch.walkers.info.cpu().numpy(),
               naccept=int(ch.naccept.item()))
    torch.cuda.synchronize()
    return rec


class _Sparse:
    def __init__(self, d):
        self.d = d

    def __getitem__(self, w):
        return self.d[w]


def run_gpu_chain(kind, orb, occ, unocc, k, K, seed, steps, device="cuda", forced=False,
                  refresh_every=0, kmax=None):
    """Run the CUDA path step by step through the C ABI."""
    ch = mc.Chain(kind, torch.as_tensor(orb, device=device), torch.as_tensor(occ, device=device),
                  torch.as_tensor(unocc, device=device), k=k, K=K, seed=seed, kmax=kmax)
    rec = record_chain(ch, steps, forced, refresh_every)
    rec["kernels"] = {c: ch.walkers.kernel_name(i) for i, c in
                      enumerate(("ratio", "update", "append", "flush", "ypass"))}
    return rec


def run_oracle(kind, orb, occ, unocc, k, seed, steps, walkers, scratch_every=1, forced=False, orb_of=None):
    """Oracle trajectories of the listed walkers (C oracle, OpenMP over walkers), immediate
    updates (delayed == immediate is the oracle's own pin).  ``forced``: xi = -1, so
    that xi < min(1,|r|^2) always holds.  ``orb_of``: walker -> its orbital matrix (when
    ``orb`` is not a host array of all walkers)."""
    W, n = occ.shape
    get = (lambda w: orb[w]) if orb_of is None else orb_of
    orbs = np.stack([get(w) for w in walkers])
    M = orbs.shape[1]
    P, J, xi = wl.proposals(seed, W, steps, n, M, k, walkers=walkers)
    if forced:
        xi = np.full_like(xi, -1.0)
    res = orc.batch(kind, orbs, np.asarray(occ)[walkers], np.asarray(unocc)[walkers], P, J, xi,
                    scratch_every=scratch_every, delay=0, final_scratch=True)
    out = {}
    for a, w in enumerate(walkers):
        out[w] = res[a]
        out[w]["P"], out[w]["J"], out[w]["xi"] = P[:, a], J[:, a], xi[:, a]
    return out


def compare(kind, rec, oracle, inv_tol=1e-9, strict=False, pure_floor=None, label=None, forced=False):
    """Element-by-element parity of one GPU record against oracle trajectories.

    Pass rule (DESIGN.md §3 reading 14).  r*_t = the oracle's from-scratch ratio,
    r_smw,t = the oracle's own naive-Woodbury ratio, e_t = max_{s<=t} |r_smw,s - r*_s|/|r*_s|
    over the from-scratch points so far (the plain fp64 algorithm's own error on this
    walker: it sits in the tracked inverse, so it persists).  Then
      * at a point with r*:      |r_gpu - r*|    <= min(1e-10 + 4 e_t, 1e-8) |r*|
      * at a point without r*:   |r_gpu - r_smw| <= min(1e-10 + 5 e_T, 1e-8) |r_smw|,
        e_T = e at the end of the trajectory (triangle inequality: the reference itself is off
        by the oracle's own error, which is only sampled at the from-scratch points)
      * ``strict`` (chains that call lrux_*_refresh): the bare 1e-10 at every point with r*.
      * ``forced`` (every proposal applied, however small its ratio -- Metropolis would never
        accept those -- so the walker runs through nearly singular matrices and the step at
        which an implementation loses its digits is implementation specific -- the oracle works
        in the paper's update-vector form, the library in the new-rows form): 8 e_T instead of
        4 e_t at every point, and the residual bound grows with e_T as well (never past 1e-7).
    ``pure_floor``: least fraction of the from-scratch points that must meet the bare
    1e-10.  Decisions must match exactly unless the oracle logged a near-tie (then the
    walker is dropped from later comparison and counted).  Returns / prints statistics:
    points, from-scratch points, fraction within the bare 1e-10, max relative error and
    |r| where it occurred, the oracle's own worst error.
    """
    st = dict(points=0, scratch_points=0, pure=0, max_rel=0.0, abs_r_at_max=0.0, e_oracle=0.0,
              dropped=0, max_inv_rel=0.0)
    for w, tr in oracle.items():
        steps = len(tr["xi"])
        assert np.array_equal(rec["idx"][:, w], tr["P"]), "proposal slots differ (RNG mismatch)"
        assert np.array_equal(rec["upos"][:, w], tr["J"]), "proposal orbitals differ (RNG mismatch)"
        assert abs(rec["init_logabs"][w] - tr["init_logabs"]) <= RTOL * max(1.0, abs(tr["init_logabs"]))
        assert abs(rec["init_phase"][w] - tr["init_phase"]) < 1e-9
        dropped = False
        e_run = 0.0
        m = ~np.isnan(tr["r_scratch"])
        e_all = float(np.max(np.abs(tr["r_lemma"][m] - tr["r_scratch"][m]) / np.abs(tr["r_scratch"][m]))) if m.any() else 0.0
        for t in range(steps):
            rg, rl, rs = rec["ratio"][t, w], tr["r_lemma"][t], tr["r_scratch"][t]
            have = not np.isnan(rs)
            ref = rs if have else rl
            if have:
                e_run = max(e_run, abs(rl - rs) / abs(rs))
            rel = abs(rg - ref) / abs(ref)
            st["points"] += 1
            if have:
                st["scratch_points"] += 1
                st["pure"] += rel <= RTOL
                if rel > st["max_rel"]:
                    st["max_rel"], st["abs_r_at_max"] = float(rel), float(abs(ref))
            bound = RTOL if (strict and have) else min(RTOL + ((8 * e_all if forced else 4 * e_run) if have else
                                                               (9 if forced else 5) * e_all), CAP)
            assert rel <= bound, ("walker %d step %d: gpu %r from-scratch %r lemma %r: rel %.3e > %.3e"
                                  % (w, t, rg, rs, rl, rel, bound))
            if bool(rec["mask"][t, w]) != bool(tr["accepted"][t]):
                assert tr["near_tie"][t], "decision mismatch at walker %d step %d" % (w, t)
                dropped = True
                st["dropped"] += 1
                break
        st["e_oracle"] = max(st["e_oracle"], e_run)
        if dropped:
            continue
        assert np.array_equal(rec["occ"][w], tr["occ"])
        assert np.array_equal(rec["unocc"][w], tr["unocc"])
        # amplitude: tracked on the GPU vs recomputed from scratch by the oracle
        if strict:
            la_tol = RTOL * max(1.0, abs(tr["scratch_logabs"]))
        else:
            la_tol = min(RTOL * max(1.0, abs(tr["scratch_logabs"]))
                         + 4 * abs(tr["logabs"] - tr["scratch_logabs"]) + 4 * e_run, CAP * max(1.0, abs(tr["scratch_logabs"])))
        assert abs(rec["logabs"][w] - tr["scratch_logabs"]) <= la_tol, (
            "walker %d: log-amplitude %r vs from-scratch %r (oracle tracked %r)"
            % (w, rec["logabs"][w], tr["scratch_logabs"], tr["logabs"]))
        assert abs(rec["phase"][w] - tr["scratch_phase"]) <= 1e-9
        n = tr["A"].shape[0]
        gi = rec["Ainv"][w]
        resid = np.abs(tr["A"] @ gi - np.eye(n)).max()
        res_tol = min(max(inv_tol, 100 * e_all), 1e-7) if forced else inv_tol
        assert resid <= res_tol, "A_T A_T^-1 residual %g" % resid
        # the inverse itself, element by element, against the oracle's tracked inverse: both
        # carry their own Woodbury error, so the bound is the residual bound in units of |A^-1|
        inv_rel = np.abs(gi - tr["Ainv"]).max() / np.abs(tr["Ainv"]).max()
        st["max_inv_rel"] = max(st["max_inv_rel"], float(inv_rel))
        assert inv_rel <= min(max(inv_tol, 50 * e_all), 1e-6), "inverse differs from the oracle's: %g" % inv_rel
        if kind == "pf":
            assert np.array_equal(gi, -gi.T), "stored inverse not exactly skew"
    st["pure_frac"] = st["pure"] / max(1, st["scratch_points"])
    if pure_floor is not None and st["scratch_points"]:
        assert st["pure_frac"] >= pure_floor, "only %.4f of the points within the bare 1e-10" % st["pure_frac"]
    report(label or kind, st)
    return st


def report(label, st):
    """Print the parity statistics (pytest -s / -rA shows them) and append them to
    gpurun_out/parity_stats.jsonl when that scratch folder exists."""
    line = ("parity[%s]: %d points (%d from scratch), within bare 1e-10: %.4f, max rel %.2e at |r| = %.2e, "
            "oracle's own worst %.2e, inverse vs oracle %.2e, dropped %d"
            % (label, st["points"], st["scratch_points"], st["pure_frac"], st["max_rel"], st["abs_r_at_max"],
               st["e_oracle"], st["max_inv_rel"], st["dropped"]))
    print(line)
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "parity_stats.jsonl"), "a") as f:
            f.write(json.dumps(dict(st, label=label), default=float) + "\n")
