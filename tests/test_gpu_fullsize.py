"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(same input generator, same chain object, same walker counts): the chain runs on every
walker; the oracle replays a few sampled walkers from the downloaded bytes of their
orbital matrices, so GPU and oracle consume identical inputs."""
import numpy as np
import pytest
import torch

import bench
import parity_util as pu
from paper_2602_05255_b200 import workload as wl

pytestmark = pytest.mark.gpu


def _record(ch, steps, sample):
    W, k = ch.W, ch.k
    ph0, la0 = ch.walkers.get_amplitude()
    rec = dict(ratio=np.zeros((steps, W), ch.ratio.cpu().numpy().dtype), mask=np.zeros((steps, W), bool),
               idx=np.zeros((steps, W, k), np.int32), upos=np.zeros((steps, W, k), np.int32),
               init_phase=ph0.cpu().numpy(), init_logabs=la0.cpu().numpy())
    for t in range(steps):
        ch.step(t)
        rec["ratio"][t] = ch.ratio.cpu().numpy()
        rec["mask"][t] = ch.mask.cpu().numpy().astype(bool)
        rec["idx"][t] = ch.idx.cpu().numpy()
        rec["upos"][t] = ch.upos.cpu().numpy()
    ph, la = ch.walkers.get_amplitude()
    n = ch.n
    full = ch.walkers.get_inverse()
    Ainv = {w: full[w].cpu().numpy() for w in sample}
    del full
    rec.update(phase=ph.cpu().numpy(), logabs=la.cpu().numpy(), occ=ch.occ.cpu().numpy(),
               unocc=ch.unocc.cpu().numpy(), info=ch.walkers.info.cpu().numpy(),
               naccept=int(ch.naccept.item()))
    rec["Ainv"] = _Sparse(Ainv)
    return rec


class _Sparse:
    def __init__(self, d):
        self.d = d

    def __getitem__(self, w):
        return self.d[w]


@pytest.mark.parametrize("name,K,steps,sample,scratch_every", [
    ("c2", 0, 40, [0, 1777, 4095], 1),       # configs[1], immediate
    ("c2", 16, 40, [5, 2048], 1),            # configs[1], delay depth 16
    ("c3", 0, 60, [0, 511, 1023], 1),        # configs[2]
    ("c4", 32, 12, [3], 0),                  # configs[3]: complex128 n=1024 (lemma-only oracle)
])
def test_full_size_config(name, K, steps, sample, scratch_every):
    wk = bench.parse_workload(name)
    W = wk["W"]
    seed, orb, occ, unocc = bench.build_inputs(wk, W, 0, torch.device("cuda"))
    bench._MASTERS.clear()
    ch = bench.make_chain(wk, K, seed, orb, occ, unocc, 0, torch.device("cuda"))
    bench._MASTERS.clear()
    rec = _record(ch, steps, sample)
    assert not rec["info"].any()
    acc = rec["mask"].mean()
    assert 0.1 < acc < 0.6, acc
    assert rec["naccept"] == rec["mask"].sum()
    orb_h = {w: orb[w].cpu().numpy() for w in sample}
    P, J, xi = wl.proposals(seed, W, steps, wk["n"], wk["M"], wk["k"], walkers=sample)
    from oracle import lrux_oracle as orc

    fn = orc.det_trajectory if wk["kind"] == "det" else orc.pf_trajectory
    oracle = {}
    for a, w in enumerate(sample):
        oracle[w] = fn(orb_h[w], occ[w], unocc[w], P[:, a], J[:, a], xi[:, a], scratch_every=scratch_every)
        oracle[w]["P"], oracle[w]["J"], oracle[w]["xi"] = P[:, a], J[:, a], xi[:, a]
    stats = pu.compare(wk["kind"], rec, oracle)
    assert stats["dropped"] == 0
