"""GPU parity: the CUDA path (through the C ABI) vs the oracle, element by element
on the same seeded inputs.  Tolerance: relative 1e-10 (BASELINE.json north_star)
with the conditioning slack of parity_util.compare; decisions exact."""
import numpy as np
import pytest
import torch

from paper_2602_05255_b200 import lrux
from paper_2602_05255_b200 import workload as wl

import parity_util as pu

pytestmark = pytest.mark.gpu


def _run(kind, seed, W, n, M, k, K, steps, cplx=False, walkers=None, scratch_every=1):
    orb, occ, unocc = pu.make_inputs(kind, seed, W, n, M, cplx)
    rec = pu.run_gpu_chain(kind, orb, occ, unocc, k, K, seed, steps)
    assert not rec["info"].any(), rec["info"]
    walkers = list(range(W)) if walkers is None else walkers
    oracle = pu.run_oracle(kind, orb, occ, unocc, k, seed, steps, walkers, scratch_every)
    stats = pu.compare(kind, rec, oracle)
    assert stats["dropped"] == 0
    acc = rec["mask"].mean()
    assert 0.05 < acc < 0.8, acc
    assert rec["naccept"] == rec["mask"].sum()
    return stats


def test_det_config1():
    """BASELINE.json configs[0]: 1 walker, n=32, M=64, k=1, 200 steps, no delay."""
    stats = _run("det", wl.BASE_SEED + 1, 1, 32, 64, 1, 0, 200)
    assert stats["points"] == 200


@pytest.mark.parametrize("n,M,k,K,cplx", [
    (32, 64, 1, 0, False),
    (50, 100, 2, 0, False),      # ragged: n not a multiple of the 64-element chunk
    (33, 70, 3, 0, False),       # odd n: scalar (VEC=1) path
    (96, 192, 4, 0, False),
    (64, 128, 8, 0, False),
    (40, 80, 2, 0, True),
    (64, 128, 4, 0, True),
    (48, 96, 1, 4, False),       # delayed, K=4
    (50, 100, 2, 3, False),
    (64, 128, 4, 2, True),
    (40, 90, 3, 5, True),
])
def test_det_small(n, M, k, K, cplx):
    _run("det", 1234 + n + k, 6, n, M, k, K, 60, cplx)


def test_det_config2_shape_reduced():
    """configs[1] shape (n=256, M=512, k=2) on 40 walkers, 60 steps; oracle on 4 of
    them; spans 4 row tiles x several waves of the update kernel."""
    for K in (0, 16):
        _run("det", wl.BASE_SEED + 2, 40, 256, 512, 2, K, 60, walkers=[0, 13, 27, 39])


@pytest.mark.parametrize("n,k", [(1101, 2), (1100, 1)])
def test_det_large_n_stream_path(n, k):
    """Large rows: n=1101 (odd: rows not 16-byte aligned) takes the generic streaming
    update kernel, n=1100 the TMA-staged one with a ragged chunk tail."""
    _run("det", 77, 3, n, 2 * n, k, 0, 12, walkers=[0, 2], scratch_every=4)


@pytest.mark.parametrize("n,M,k,K,cplx", [
    (32, 64, 1, 0, False),
    (50, 100, 1, 0, False),
    (64, 128, 1, 0, False),      # register-resident kernel, n = 64 instance
    (34, 70, 2, 0, False),
    (64, 128, 3, 0, False),
    (40, 80, 4, 0, False),
    (32, 64, 1, 0, True),
    (36, 72, 2, 0, True),
    (48, 96, 1, 4, False),
    (50, 100, 2, 3, False),
    (32, 64, 2, 2, True),
])
def test_pf_small(n, M, k, K, cplx):
    _run("pf", 4321 + n + k, 6, n, M, k, K, 60, cplx)


def test_pf_config3_shape_reduced():
    """configs[2] shape (n=128, M=256, k=1) on 24 walkers, 80 steps; oracle on 4."""
    _run("pf", wl.BASE_SEED + 3, 24, 128, 256, 1, 0, 80, walkers=[0, 7, 15, 23])


@pytest.mark.parametrize("n,k,K,cplx,steps", [
    (1024, 4, 0, False, 10),     # rows of 8 KB: RC=4 rows per bulk copy, 2 vectors per lane
    (1024, 8, 0, False, 8),      # k=8: 32 partial sums per warp
    (1100, 1, 0, False, 10),     # ragged: 550 vectors per row, 4-row chunks with a 3-row tail
    (512, 2, 0, True, 10),       # complex128, 8 KB rows
    (2048, 2, 0, False, 4),      # 16 KB rows: RC=2, 4 vectors per lane
    (1100, 8, 0, False, 8),      # no rank-8 instance at this n: split into two rank-4 passes
    (1100, 7, 0, False, 8),      # 4 + 3
    (1024, 2, 3, False, 14),     # delayed append through the same pass + finish kernel
    (512, 4, 2, True, 12),       # complex128 delayed (configs[3] shape at n=512)
])
def test_det_tma_update_path(n, k, K, cplx, steps):
    """Immediate update / delayed append through the TMA-staged kernel (lrux_det_tma.cu).
    The delayed variant is opt-in (LRUX_UPDATE_PATH=tma), see launch_append_kt."""
    import os

    old = os.environ.get("LRUX_UPDATE_PATH")
    if K > 0:
        os.environ["LRUX_UPDATE_PATH"] = "tma"
    try:
        _run("det", 500 + n + k, 2, n, 2 * n, k, K, steps, cplx, walkers=[1],
             scratch_every=0 if n >= 2048 else steps - 1)
    finally:
        if K > 0:
            if old is None:
                del os.environ["LRUX_UPDATE_PATH"]
            else:
                os.environ["LRUX_UPDATE_PATH"] = old


def test_det_tma_update_n4096_properties():
    """n=4096 (32 KB rows, one row per bulk copy): the oracle is too slow here, so check
    what holds at any size: A_T A_T^-1 = 1 and the tracked amplitude against a library
    slogdet of A_T."""
    from paper_2602_05255_b200 import mc

    n, M, W, k = 4096, 8192, 2, 2
    seed = 4242
    Phi = wl.orbital_matrices_torch(seed, 0, W, M, n, 1.0 / n, "cuda")
    occ, unocc = wl.initial_occupations(seed, W, M, n)
    ch = mc.Chain("det", Phi, torch.as_tensor(occ, device="cuda"), torch.as_tensor(unocc, device="cuda"),
                  k=k, K=0, seed=seed)
    for t in range(8):
        ch.step(t, forced=(t % 2 == 0))
    torch.cuda.synchronize()
    assert not ch.walkers.info.any()
    assert int(ch.naccept.item()) >= 4 * W
    ph, la = ch.walkers.get_amplitude()
    inv = ch.walkers.get_inverse()
    for w in range(W):
        A = Phi[w][ch.occ[w].long()]
        resid = (A @ inv[w] - torch.eye(n, dtype=A.dtype, device="cuda")).abs().max().item()
        assert resid < 1e-9, resid
        sign, logabs = torch.linalg.slogdet(A)
        assert abs(la[w].item() - logabs.item()) < 1e-8 * max(1.0, abs(logabs.item()))
        assert ph[w].item() == sign.item()


@pytest.mark.parametrize("n,k", [(200, 1), (200, 2), (320, 1), (320, 2)])
def test_pf_large_n_paths(n, k):
    """n=200: the inverse (320 KB) does not fit in one CTA's shared memory -> 8-CTA cluster
    kernels (row slabs, Y over DSMEM); n=320: beyond the cluster kernels too -> Y pass +
    streaming update."""
    _run("pf", 99 + k, 3, n, 2 * n, k, 0, 10, walkers=[0, 2], scratch_every=3)


@pytest.mark.parametrize("path", ["smem", "nb5", "cluster", "cluster_generic", "cta"])
def test_pf_config3_shape_older_kernels(path, monkeypatch):
    """The Pfaffian update kernels the register-resident one superseded at n = 128 stay
    selectable (LRUX_PF_PATH, read at every accept) and must give the same trajectory:
    shared-memory resident with 6 / 5 chunk buffers, 4-CTA cluster column-pair kernel,
    generic cluster kernel, single-CTA warp-per-row kernel."""
    monkeypatch.setenv("LRUX_PF_PATH", path)
    _run("pf", wl.BASE_SEED + 3, 12, 128, 256, 1, 0, 40, walkers=[0, 5, 11])


def test_det_config4_shape_reduced():
    """configs[3] shape reduced: complex128, k=4, delay K=32, n=256."""
    _run("det", wl.BASE_SEED + 4, 6, 256, 512, 4, 32, 80, cplx=True, walkers=[0, 5], scratch_every=5)


def test_attach_resumes_from_a_state_copy():
    """lrux_*_attach: a byte copy of the state buffer is a checkpoint; a chain resumed
    from it reproduces the original chain bit for bit (det with a half-full delay
    buffer, and Pfaffian)."""
    from paper_2602_05255_b200 import mc

    for kind, n, M, k, K in (("det", 48, 96, 2, 5), ("pf", 40, 80, 1, 0)):
        seed = 31 + n
        orb, occ, unocc = pu.make_inputs(kind, seed, 5, n, M)
        dev = "cuda"
        a = mc.Chain(kind, torch.as_tensor(orb, device=dev), torch.as_tensor(occ, device=dev),
                     torch.as_tensor(unocc, device=dev), k=k, K=K, seed=seed)
        for t in range(7):
            a.step(t)
        b = mc.Chain(kind, a.orb, a.occ.clone(), a.unocc.clone(), k=k, K=K, seed=seed,
                     walkers=a.walkers.clone())
        for t in range(7, 20):
            a.step(t)
            b.step(t)
            assert torch.equal(a.ratio, b.ratio) and torch.equal(a.mask, b.mask)
        assert torch.equal(a.walkers.get_inverse(), b.walkers.get_inverse())
        pa, la = a.walkers.get_amplitude()
        pb, lb = b.walkers.get_amplitude()
        assert torch.equal(pa, pb) and torch.equal(la, lb)


# ---------------------------------------------------------------- error paths
def test_errors_and_info_bits():
    dev = "cuda"
    W, n = 4, 16
    rng = np.random.default_rng(3)
    A0 = rng.standard_normal((W, n, n))
    A0[2] = 0.0                                           # singular walker
    wk = lrux.DetWalkers(torch.as_tensor(A0, device=dev), kmax=2, K=0)
    torch.cuda.synchronize()
    assert wk.info.cpu().tolist() == [0, 0, 1, 0]
    mask = torch.ones(W, dtype=torch.uint8, device=dev)
    with pytest.raises(lrux.LruxError) as e:              # accept without pending ratio
        wk.accept(mask)
    assert e.value.status == lrux.ESTATE
    idx = torch.tensor([[0, 1], [3, 3], [0, 1], [0, 99]], dtype=torch.int32, device=dev)
    rows = torch.as_tensor(rng.standard_normal((W, 2, n)), device=dev)
    r = wk.ratio_(idx, rows).cpu().numpy()
    assert np.isfinite(r[0]) and np.isnan(r[1]) and np.isnan(r[3])
    inv_before = wk.get_inverse().cpu().numpy()
    wk.ratio_(idx, rows)
    wk.accept(mask)
    info = wk.info.cpu().numpy()
    assert info[0] == 0 and (info[1] & 2) and (info[3] & 2)
    inv_after = wk.get_inverse().cpu().numpy()
    assert not np.array_equal(inv_after[0], inv_before[0])          # walker 0 moved
    assert np.array_equal(inv_after[1], inv_before[1])              # bad proposals left untouched
    assert np.array_equal(inv_after[3], inv_before[3])
    with pytest.raises(lrux.LruxError):                   # k > kmax
        wk.ratio_(torch.zeros((W, 3), dtype=torch.int32, device=dev),
                  torch.zeros((W, 3, n), dtype=torch.float64, device=dev))
    with pytest.raises(lrux.LruxError):                   # odd n for a Pfaffian
        lrux.PfWalkers(torch.zeros((2, 5, 5), dtype=torch.float64, device=dev))


@pytest.mark.parametrize("kind,n,cplx", [("det", 800, False), ("det", 1000, False),
                                          ("det", 800, True), ("pf", 1000, False)])
def test_blocked_init(kind, n, cplx):
    """Step a0 through the blocked (panel + DMMA) Gauss-Jordan path (n >= 768), including a
    ragged last panel (1000 = 31*32 + 8), a walker that needs row exchanges in every panel
    and a singular walker."""
    from oracle import lrux_oracle as orc

    rng = np.random.default_rng(n + cplx)
    W = 3
    A = rng.standard_normal((W, n, n))
    if cplx:
        A = A + 1j * rng.standard_normal((W, n, n))
    if kind == "pf":
        A = np.triu(A, 1) - np.triu(A, 1).transpose(0, 2, 1)
    else:
        A[1] = A[1][rng.permutation(n)] * 1e-3       # pivots far from the diagonal, small scale
        A[2, 5] = 0.0                                 # a zero row: exactly singular
    wk = (lrux.DetWalkers if kind == "det" else lrux.PfWalkers)(torch.as_tensor(A, device="cuda"), kmax=1)
    ph, la = wk.get_amplitude()
    inv = wk.get_inverse().cpu().numpy()
    info = wk.info.cpu().numpy()
    good = [0, 1] if kind == "det" else [0, 1, 2]
    if kind == "det":
        assert info[2] & 1 and np.isneginf(la[2].item())
    for w in good:
        assert info[w] == 0
        oph, ola = orc.slogdet(A[w]) if kind == "det" else orc.slogpf(A[w])
        assert abs(ph[w].item() - oph) < 1e-9
        assert abs(la[w].item() - ola) <= 1e-10 * max(1.0, abs(ola))
        assert np.abs(inv[w] @ A[w] - np.eye(n)).max() < 1e-7
        if kind == "pf":
            assert np.array_equal(inv[w], -inv[w].T)


def test_init_amplitude_and_inverse():
    """Step a0 alone: A^-1 and (phase, log|det|), (phase, log|pf|) vs the oracle."""
    from oracle import lrux_oracle as orc

    rng = np.random.default_rng(11)
    for cplx in (False, True):
        for n in (1, 2, 7, 64, 130):
            A = rng.standard_normal((3, n, n))
            if cplx:
                A = A + 1j * rng.standard_normal((3, n, n))
            wk = lrux.DetWalkers(torch.as_tensor(A, device="cuda"), kmax=1)
            ph, la = wk.get_amplitude()
            inv = wk.get_inverse().cpu().numpy()
            for w in range(3):
                oph, ola = orc.slogdet(A[w])
                assert abs(ph[w].item() - oph) < 1e-9
                assert abs(la[w].item() - ola) <= 1e-10 * max(1.0, abs(ola))
                assert np.abs(inv[w] @ A[w] - np.eye(n)).max() < 1e-8
        for n in (2, 8, 64, 130):
            g = rng.standard_normal((3, n, n))
            if cplx:
                g = g + 1j * rng.standard_normal((3, n, n))
            A = np.triu(g, 1) - np.triu(g, 1).transpose(0, 2, 1)
            wk = lrux.PfWalkers(torch.as_tensor(A, device="cuda"), kmax=1)
            ph, la = wk.get_amplitude()
            inv = wk.get_inverse().cpu().numpy()
            for w in range(3):
                oph, ola = orc.slogpf(A[w])
                assert abs(ph[w].item() - oph) < 1e-9
                assert abs(la[w].item() - ola) <= 1e-10 * max(1.0, abs(ola))
                assert np.abs(inv[w] @ A[w] - np.eye(n)).max() < 1e-8
                assert np.array_equal(inv[w], -inv[w].T)
