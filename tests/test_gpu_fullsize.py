"""Parity at BASELINE.json's FULL sizes over the FULL trajectories, in the launch
configuration bench.py times (same input generator, same chain object, same walker
counts): the chain runs on every walker for every step of the config (1000 / 1000 / 500);
the oracle replays a few sampled walkers from the downloaded bytes of their orbital
matrices, so GPU and oracle consume identical inputs."""
import numpy as np
import pytest
import torch

import bench
import parity_util as pu

pytestmark = pytest.mark.gpu


def _chain(name, K):
    wk = bench.parse_workload(name)
    seed, orb, occ, unocc = bench.build_inputs(wk, wk["W"], 0, torch.device("cuda"))
    bench._MASTERS.clear()
    ch = bench.make_chain(wk, K, seed, orb, occ, unocc, 0, torch.device("cuda"))
    bench._MASTERS.clear()
    return wk, seed, orb, occ, unocc, ch


@pytest.mark.parametrize("name,K,steps,sample,scratch_every,pure_floor", [
    # pure_floor: least fraction of the from-scratch points within the BARE 1e-10 (measured on
    # B200 in round 2: 1.0000 / 0.9980 / 1.0000 / 1.0000)
    ("c2", 0, 1000, [0, 1777, 4095], 1, 0.99),    # configs[1], immediate, all 1000 steps
    ("c2", 16, 1000, [5, 2048], 1, 0.99),         # configs[1], delay depth 16
    ("c3", 0, 1000, [0, 511, 1023], 1, 0.99),     # configs[2], all 1000 steps
    ("c4", 32, 500, [3, 300], 25, 0.99),          # configs[3], all 500 steps; from scratch every 25th
])
def test_full_size_full_trajectory(name, K, steps, sample, scratch_every, pure_floor):
    wk, seed, orb, occ, unocc, ch = _chain(name, K)
    rec = pu.record_chain(ch, steps, sample=sample)
    assert not rec["info"].any()
    acc = rec["mask"].mean()
    assert 0.1 < acc < 0.6, acc
    assert rec["naccept"] == rec["mask"].sum()
    oracle = pu.run_oracle(wk["kind"], None, occ, unocc, wk["k"], seed, steps, sample, scratch_every,
                           orb_of=lambda w: orb[w].cpu().numpy())
    stats = pu.compare(wk["kind"], rec, oracle, pure_floor=pure_floor,
                       label="%s K=%d full size, %d steps" % (name, K, steps))
    assert stats["dropped"] == 0 and stats["points"] == steps * len(sample)


def test_c4_full_depth_flush_at_full_size():
    """configs[3]'s own flush: complex128, n = 1024, k = 4, K = 32 -- the automatic fold at
    full depth (K k = 128 columns, 8 chunks of the complex staging loop) fires after 32
    applied updates; 35 forced steps, flushed inverse compared element by element."""
    wk, seed, orb, occ, unocc, ch = _chain("c4", 32)
    sample = [7]
    f0 = ch.walkers.flush_count()
    rec = pu.record_chain(ch, 35, forced=True, sample=sample)
    f1 = ch.walkers.flush_count()
    assert f1[0] - f0[0] >= wk["W"] and f1[1] - f0[1] >= wk["W"] * 128     # every walker folded 128 columns
    assert ch.walkers.kernel_name(3) == "flush_dmma_kernel"
    oracle = pu.run_oracle("det", None, occ, unocc, wk["k"], seed, 35, sample, 34, forced=True,
                           orb_of=lambda w: orb[w].cpu().numpy())
    stats = pu.compare("det", rec, oracle, label="c4 forced 35 steps, full-depth flush", forced=True)
    assert stats["max_inv_rel"] < 1e-9
