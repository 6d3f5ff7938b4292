"""Stream-ordered Metropolis chains driving the C-ABI library (harness level).

One step = lruxh_*_propose -> lrux_*_ratio -> lruxh_decide -> lrux_*_accept, all
enqueued on the current CUDA stream without host synchronisation.  This is the
"step" bench.py times and the parity tests replay against the oracle.
"""
from __future__ import annotations

import torch

from . import lrux


class Chain:
    """Determinant (orbitals=Phi [W][M][n]) or Pfaffian (orbitals=F [W][M][M]) chain.

    occ [W][n], unocc [W][M-n] int32 device tensors are updated in place.
    """

    def __init__(self, kind, orbitals, occ, unocc, k, K=0, seed=0, w0=0, kmax=None, walkers=None, guard=0):
        assert kind in ("det", "pf")
        self.kind, self.k, self.K, self.seed, self.w0 = kind, int(k), int(K), int(seed), int(w0)
        self.orb = orbitals.contiguous()
        self.occ = occ.to(torch.int32).contiguous()
        self.unocc = unocc.to(torch.int32).contiguous()
        dev, dt = self.orb.device, self.orb.dtype
        self.W, self.n = self.occ.shape
        self.M = self.orb.shape[1]
        W, n = self.W, self.n
        if walkers is not None:       # already initialised (e.g. a clone of the step-0 state)
            self.walkers = walkers
            self._buffers(W, n, dt, dev)
            return
        A0 = torch.empty((W, n, n), dtype=dt, device=dev)
        step = max(1, (1 << 26) // (n * n))        # bound the temporaries of the index gather
        for c0 in range(0, W, step):
            c1 = min(W, c0 + step)
            ar = torch.arange(c0, c1, device=dev)[:, None]
            occl = self.occ[c0:c1].long()
            if kind == "det":
                A0[c0:c1] = self.orb[ar, occl]                        # Phi[w][occ,:]
            else:
                A0[c0:c1] = self.orb[ar[:, :, None], occl[:, :, None], occl[:, None, :]]
        cls = lrux.DetWalkers if kind == "det" else lrux.PfWalkers
        self.walkers = cls(A0, kmax=self.k if kmax is None else kmax, K=self.K, guard=guard)
        del A0
        self._buffers(W, n, dt, dev)

    def _buffers(self, W, n, dt, dev):
        self.idx = torch.zeros((W, self.k), dtype=torch.int32, device=dev)
        self.upos = torch.zeros((W, self.k), dtype=torch.int32, device=dev)
        self.rows = torch.zeros((W, self.k, n), dtype=dt, device=dev)
        self.mask = torch.zeros(W, dtype=torch.uint8, device=dev)
        self.naccept = torch.zeros(1, dtype=torch.int64, device=dev)
        self.ratio = self.walkers.ratio
        # |r|^2 = 4 -> the Metropolis test always passes: forced-accept mode
        self.force_ratio = torch.full((W,), 2.0, dtype=dt, device=dev)
        self.harness_launches = 0

    def propose(self, t, d_step=None):
        fn = lrux.det_propose if self.kind == "det" else lrux.pf_propose
        fn(self.seed, self.w0, t, self.orb, self.occ, self.unocc, self.idx, self.upos, self.rows, d_step)
        self.harness_launches += 1

    def step(self, t, forced=False, d_step=None):
        """One Monte-Carlo step of every walker.  ``forced``: every proposal with a
        regular R is applied (what the paper's Fig. 2 times)."""
        self.propose(t, d_step)
        self.walkers.ratio_(self.idx, self.rows)
        lrux.decide(self.seed, self.w0, t, self.force_ratio if forced else self.ratio, self.idx,
                    self.upos, self.occ, self.unocc, self.mask, self.naccept, d_step)
        self.harness_launches += 1
        self.walkers.accept(self.mask)

    def capture(self, t_next, forced=False):
        """Capture ONE step (propose -> ratio -> decide -> accept) into a CUDA graph whose step
        number lives in device memory; ``replay()`` then runs step t_next, t_next + 1, ... with
        a single host call each.  The launch sequence of a step depends on the shape only and no
        call synchronises, so the replayed chain is the stream-launched chain, kernel for kernel.
        Run at least one eager step first (kernel attributes are configured on first use)."""
        self.d_step = torch.tensor([int(t_next), 0], dtype=torch.int64, device=self.occ.device)
        l0 = self.launches()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph):
            self.step(0, forced, self.d_step)
        self.launches_per_replay = self.launches() - l0      # enqueued while capturing, run by every replay
        self.replays = 0
        return self.graph

    def replay(self):
        self.graph.replay()
        self.replays += 1

    def launches(self):
        """Kernel launches enqueued by stream calls (a captured step counts once, at capture)."""
        return self.walkers.launch_count() + self.harness_launches
