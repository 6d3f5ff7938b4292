"""Helpers for the GPU-vs-oracle parity tests (tests only)."""
import numpy as np
import torch

from oracle import lrux_oracle as orc
from paper_2602_05255_b200 import mc
from paper_2602_05255_b200 import workload as wl

RTOL = 1e-10   # BASELINE.json north_star: relative 1e-10 on ratios and log-amplitudes


def make_inputs(kind, seed, W, n, M, cplx=False):
    """Host-generated inputs (identical bytes go to the GPU and to the oracle)."""
    if kind == "det":
        var = 1.0 / (2 * n) if cplx else 1.0 / n
        orb = np.stack([wl.orbital_matrix(seed, w, M, n, var, cplx) for w in range(W)])
    else:
        orb = np.stack([wl.pairing_matrix(seed, w, M, 1.0 / n, cplx) for w in range(W)])
    occ, unocc = wl.initial_occupations(seed, W, M, n)
    return orb, occ, unocc


def run_gpu_chain(kind, orb, occ, unocc, k, K, seed, steps, device="cuda"):
    """Run the CUDA path step by step, recording ratio and mask of every step."""
    ch = mc.Chain(kind, torch.as_tensor(orb, device=device), torch.as_tensor(occ, device=device),
                  torch.as_tensor(unocc, device=device), k=k, K=K, seed=seed)
    W = orb.shape[0]
    ph0, la0 = ch.walkers.get_amplitude()
    rec = dict(ratio=np.zeros((steps, W), orb.dtype), mask=np.zeros((steps, W), bool),
               idx=np.zeros((steps, W, k), np.int32), upos=np.zeros((steps, W, k), np.int32),
               init_phase=ph0.cpu().numpy(), init_logabs=la0.cpu().numpy())
    for t in range(steps):
        ch.step(t)
        rec["ratio"][t] = ch.ratio.cpu().numpy()
        rec["mask"][t] = ch.mask.cpu().numpy().astype(bool)
        rec["idx"][t] = ch.idx.cpu().numpy()
        rec["upos"][t] = ch.upos.cpu().numpy()
    ph, la = ch.walkers.get_amplitude()
    rec.update(phase=ph.cpu().numpy(), logabs=la.cpu().numpy(),
               Ainv=ch.walkers.get_inverse().cpu().numpy(), occ=ch.occ.cpu().numpy(),
               unocc=ch.unocc.cpu().numpy(), info=ch.walkers.info.cpu().numpy(),
               naccept=int(ch.naccept.item()))
    torch.cuda.synchronize()
    return rec


def run_oracle(kind, orb, occ, unocc, k, seed, steps, walkers, scratch_every=1):
    W, n = occ.shape
    M = orb.shape[1]
    P, J, xi = wl.proposals(seed, W, steps, n, M, k, walkers=walkers)
    fn = orc.det_trajectory if kind == "det" else orc.pf_trajectory
    out = {}
    for a, w in enumerate(walkers):
        out[w] = fn(orb[w], occ[w], unocc[w], P[:, a], J[:, a], xi[:, a], scratch_every=scratch_every)
        out[w]["P"], out[w]["J"], out[w]["xi"] = P[:, a], J[:, a], xi[:, a]
    return out


def compare(kind, rec, oracle, inv_tol=1e-9):
    """Element-by-element parity of one GPU record against oracle trajectories.

    Pass rule (SURVEY.md §8(c) item 14 as read in DESIGN.md §3 reading 14): with
    r*_t the from-scratch ratio, r_smw,t the oracle's own naive-Woodbury ratio and
    e_t = max_{s<=t} |r_smw,s - r*_s| / |r*_s| the worst relative error the plain
    fp64 algorithm has shown on this walker so far (the error sits in the tracked
    inverse, so it persists after the step that exposed it),
        |r_gpu,t - r*_t| <= (1e-10 + 4 e_t) |r*_t|
    i.e. 1e-10, or no worse than 4x the plain algorithm's own error where the
    trajectory is ill-conditioned.  Decisions must match exactly unless the
    oracle logged a near-tie (then the walker is dropped from later comparison).
    Returns statistics for reporting (``pure`` counts points within the bare 1e-10).
    """
    stats = dict(points=0, pure=0, max_rel=0.0, dropped=0)
    for w, tr in oracle.items():
        steps = len(tr["xi"])
        assert np.array_equal(rec["idx"][:, w], tr["P"]), "proposal slots differ (RNG mismatch)"
        assert np.array_equal(rec["upos"][:, w], tr["J"]), "proposal orbitals differ (RNG mismatch)"
        assert rec["init_logabs"][w] == _approx(tr["init_logabs"], 1e-10 * max(1.0, abs(tr["init_logabs"])))
        assert abs(rec["init_phase"][w] - tr["init_phase"]) < 1e-9
        dropped = False
        e_run = 0.0
        for t in range(steps):
            rg, rl, rs = rec["ratio"][t, w], tr["r_lemma"][t], tr["r_scratch"][t]
            ref = rl if np.isnan(rs) else rs
            if not np.isnan(rs):
                e_run = max(e_run, abs(rl - rs) / abs(rs))
            slack = 4 * e_run * abs(ref)
            err = abs(rg - ref)
            stats["points"] += 1
            rel = err / abs(ref)
            stats["max_rel"] = max(stats["max_rel"], rel)
            stats["pure"] += rel <= RTOL
            assert err <= RTOL * abs(ref) + slack + (4e-10 * abs(ref) if np.isnan(rs) else 0.0), (
                "walker %d step %d: gpu %r oracle %r (lemma %r)" % (w, t, rg, rs, rl))
            if bool(rec["mask"][t, w]) != bool(tr["accepted"][t]):
                assert tr["near_tie"][t], "decision mismatch at walker %d step %d" % (w, t)
                dropped = True
                stats["dropped"] += 1
                break
        if dropped:
            continue
        assert np.array_equal(rec["occ"][w], tr["occ"])
        assert np.array_equal(rec["unocc"][w], tr["unocc"])
        # amplitude: tracked on the GPU vs recomputed from scratch by the oracle
        la_tol = (RTOL * max(1.0, abs(tr["scratch_logabs"])) + 4 * abs(tr["logabs"] - tr["scratch_logabs"])
                  + 4 * e_run)
        assert abs(rec["logabs"][w] - tr["scratch_logabs"]) <= la_tol
        assert abs(rec["phase"][w] - tr["scratch_phase"]) <= 1e-9
        n = tr["A"].shape[0]
        resid = np.abs(tr["A"] @ rec["Ainv"][w] - np.eye(n)).max()
        assert resid <= inv_tol, "A_T A_T^-1 residual %g" % resid
        if kind == "pf":
            assert np.array_equal(rec["Ainv"][w], -rec["Ainv"][w].T), "stored inverse not exactly skew"
    return stats


def _approx(x, tol):
    import pytest

    return pytest.approx(x, abs=tol)
