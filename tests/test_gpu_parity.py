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


def _run(kind, seed, W, n, M, k, K, steps, cplx=False, walkers=None, scratch_every=1, forced=False,
         refresh_every=0, strict=False, pure_floor=None, acc_range=(0.05, 0.8), kernel=None, kmax=None):
    orb, occ, unocc = pu.make_inputs(kind, seed, W, n, M, cplx)
    rec = pu.run_gpu_chain(kind, orb, occ, unocc, k, K, seed, steps, forced=forced,
                           refresh_every=refresh_every, kmax=kmax)
    assert not rec["info"].any(), rec["info"]
    walkers = list(range(W)) if walkers is None else walkers
    oracle = pu.run_oracle(kind, orb, occ, unocc, k, seed, steps, walkers, scratch_every, forced=forced)
    label = "%s %s n=%d k=%d K=%d%s%s" % (kind, "c128" if cplx else "f64", n, k, K,
                                         " forced" if forced else "", " refresh/%d" % refresh_every if refresh_every else "")
    if pure_floor is None and not forced:
        pure_floor = 0.95      # measured on B200: >= 0.98 on every Metropolis chain of this file
    stats = pu.compare(kind, rec, oracle, strict=strict, pure_floor=pure_floor, label=label, forced=forced)
    assert stats["dropped"] == 0
    acc = rec["mask"].mean()
    if forced:
        assert acc == 1.0
    else:
        assert acc_range[0] < acc < acc_range[1], acc
    assert rec["naccept"] == rec["mask"].sum()
    if kernel:       # the kernel this shape is meant to reach (selected by shape alone)
        for cls, name in kernel.items():
            assert name in rec["kernels"][cls], rec["kernels"]
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


@pytest.mark.parametrize("n,k,K,cplx,steps,kernel", [
    (1024, 4, 0, False, 10, "det_update_dmma_kernel"),   # real, k >= 3: 8-row strips on the FP64 tensor pipe
    (1024, 8, 0, False, 8, "det_update_dmma_kernel"),
    (1100, 8, 0, False, 8, "det_update_dmma_kernel"),    # n > 1024: columns split over a 2-CTA cluster, ragged
    (1100, 7, 0, False, 8, "det_update_dmma_kernel"),
    (2048, 8, 0, False, 4, "det_update_dmma_kernel"),    # 2-CTA cluster, even split
    (2048, 4, 0, False, 4, "det_update_tma_kernel"),     # the one rank-4 shape where the TMA-staged kernel is faster
    (500, 3, 0, False, 10, "det_update_dmma_kernel"),    # ragged last 8-column block and last strip
    (1100, 1, 0, False, 10, "det_update_tma_kernel"),    # ragged: 550 vectors per row, 4-row chunks with a 3-row tail
    (512, 2, 0, True, 10, "det_update_tma_kernel"),      # complex128, 8 KB rows
    (2048, 2, 0, False, 4, "det_update_tma_kernel"),     # 16 KB rows: RC=2, 4 vectors per lane
    (512, 8, 0, True, 8, "det_update_tma_kernel"),       # complex k=8: no rank-8 instance -> two rank-4 passes (det_split_prep_kernel)
    (1024, 2, 3, False, 14, "det_append_stream_real_kernel"),   # delayed, real rows of 8 KB
    (256, 2, 3, False, 14, "det_append_kernel"),         # n < 512 with k <= 2: the register-row pass stays (configs[1] with a delay)
    (512, 4, 2, True, 12, "det_append_kernel"),          # complex128 delayed (configs[3] shape at n=512)
])
def test_det_large_row_paths(n, k, K, cplx, steps, kernel):
    """Immediate update / delayed append at rows >= 8 KB: each shape reaches the kernel named
    (selected by shape alone) and follows the oracle."""
    _run("det", 500 + n + k, 2, n, 2 * n, k, K, steps, cplx, walkers=[1],
         scratch_every=1 if n <= 1100 else steps - 1, acc_range=(0.0, 1.0),
         kernel={"update" if K == 0 else "append": kernel})


@pytest.mark.parametrize("n,k", [(64, 4), (128, 8), (100, 3), (34, 5), (128, 4), (256, 8), (200, 5)])
def test_det_update_dmma_warp_strips(n, k):
    """Real k >= 3 at n <= 256: one warp owns a whole 8-row strip (det_update_dmma_warp_kernel);
    n = 100 / 34: ragged last block and last strip, strips of two walkers in one CTA's range."""
    _run("det", 6400 + n + k, 5, n, 2 * n, k, 0, 12, walkers=[0, 2, 4], scratch_every=1, forced=(k > 4),
         acc_range=(0.0, 1.0), kernel={"update": "det_update_dmma_warp_kernel"})


@pytest.mark.parametrize("n,k,K,cplx,name", [
    (64, 1, 0, False, "det_ratio_warp_kernel"),    # n <= 128: one warp per walker, 8 walkers per CTA
    (128, 4, 0, False, "det_ratio_warp_kernel"),
    (100, 3, 0, False, "det_ratio_warp_kernel"),   # ragged: 100 = 3 x 32 + 4 columns
    (33, 2, 0, True, "det_ratio_warp_kernel"),     # complex, odd n
    (96, 2, 4, False, "det_ratio_warp_kernel"),    # with a delay buffer: k <= 2
    (256, 2, 0, False, "det_ratio_warp_kernel"),   # configs[1] shape: n <= 256, k <= 2, no delay buffer
    (256, 2, 4, False, "det_ratio_kernel"),        # ... with a delay buffer: one CTA per walker
    (64, 4, 4, False, "det_ratio_kernel"),         # k = 4 with a delay buffer, and k = 8: one CTA per walker
    (64, 8, 0, False, "det_ratio_kernel"),
])
def test_det_ratio_kernel_by_shape(n, k, K, cplx, name):
    """The two determinant ratio kernels, each reached by its shape and checked by name."""
    _run("det", 7100 + n + k + K, 9, n, 2 * n, k, K, 30, cplx, walkers=[0, 4, 8], scratch_every=1,
         forced=(k == 8), acc_range=(0.0, 1.0), kernel={"ratio": name})


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


@pytest.mark.parametrize("n,k,cplx,name", [
    (64, 1, False, "pf_regs_k1_kernel"),          # walker in registers
    (100, 1, False, "pf_resident_k1_kernel"),     # whole walker in one CTA's shared memory, 6 chunk buffers
    (140, 1, False, "pf_resident_k1_kernel"),     # ... 5 chunk buffers
    (200, 1, False, "pf_cluster_k1_kernel"),      # 8-CTA cluster, run-time sizes
    (256, 1, False, "pf_cluster_k1_kernel"),      # 8-CTA cluster, unrolled instance
    (128, 2, False, "pf_update_dmma_warp_kernel"),    # real k >= 2, n <= 128: warp-owned 8-row strips on the FP64 tensor pipe
    (136, 2, False, "pf_update_dmma_kernel"),     # n > 128: strips split over the 8 warps
    (64, 1, True, "pf_cluster_update_kernel"),    # complex: generic cluster kernel, 4-CTA
    (128, 2, True, "pf_cluster_update_kernel"),   # ... 8-CTA, k = 2
    (96, 1, True, "pf_cluster_update_kernel"),
    (320, 1, False, "pf_update_dmma_kernel"),     # k = 1 beyond the cluster kernels: Y pass + DMMA strips (1 DMMA / block)
    (320, 2, True, "pf_update_stream_kernel"),    # complex: Y pass + streaming update
    (34, 2, False, "pf_update_dmma_warp_kernel"), # ragged: n not a multiple of 8, strips of two walkers in one range
    (520, 2, False, "pf_update_dmma_kernel"),     # 16 warps
])
def test_pf_update_kernel_by_shape(n, k, cplx, name):
    """Every immediate Pfaffian update kernel, reached by its SHAPE (there is no environment
    switch): same trajectory as the oracle."""
    _run("pf", 171 + n + k, 4, n, 2 * n, k, 0, 24, cplx, walkers=[0, 3], scratch_every=4,
         kernel={"update": name})


@pytest.mark.parametrize("n,k", [
    (250, 3),      # 2k = 6 padded to 8
    (256, 4),      # 2 DMMAs per block, 4 blocks per warp
    (130, 8),      # 2k = 16: 4 DMMAs per block
    (512, 4),      # 8 blocks per warp (the shape VERDICT r1 item 7 names)
    (64, 4),       # n <= 128: warp-owned strips (pf_update_dmma_warp_kernel), 8 blocks, prefetched
    (128, 8),      # ... 16 blocks, 4 DMMAs per block
    (100, 3),      # ... ragged
])
def test_pf_update_dmma_larger_ranks(n, k):
    """pf_update_dmma_kernel with 2 and 4 DMMAs per 8 x 8 block, every proposal applied (rank >= 3
    proposals are rarely accepted by the Metropolis test); the stored inverse must stay EXACTLY
    skew (parity_util.compare checks Ti == -Ti^T bit for bit)."""
    _run("pf", 1900 + n + k, 3, n, 2 * n, k, 0, 8, walkers=[0, 2], scratch_every=2, forced=True,
         kernel={"update": "pf_update_dmma_warp_kernel" if n <= 128 else "pf_update_dmma_kernel"})


@pytest.mark.parametrize("n,k,steps", [
    (1040, 1, 5),      # two column ranges of 520: A fragments formed from the pending area
    (1024, 8, 4),      # 2k = 16: the y, g panels of 1024 columns exceed shared memory -> two ranges of 512
    (1500, 2, 4),      # ragged ranges (752 + 748)
])
def test_pf_update_dmma_column_ranges(n, k, steps):
    """pf_update_dmma_kernel with the columns cut into ranges (n > 1024, or 2k x n panels beyond
    shared memory): a strip's own y, g rows may lie in another CTA's range; exact skewness across
    ranges (mirrored elements are produced by different CTAs)."""
    _run("pf", 1813 + n + k, 2, n, 2 * n, k, 0, steps, walkers=[1], scratch_every=4, forced=True,
         kernel={"update": "pf_update_dmma_kernel"})


def test_pf_update_tile_kernel_large_k():
    """Complex data with 4 k n e > 160 KB (n = 1024, k = 4): Y' and g no longer fit in shared
    memory -> the 32x32-tile kernel.  Forced accept."""
    _run("pf", 1812, 2, 1024, 2048, 4, 0, 3, cplx=True, walkers=[1], scratch_every=3, forced=True,
         kernel={"update": "pf_update_kernel"})


@pytest.mark.parametrize("kind,n,k,K,cplx", [
    ("det", 192, 8, 8, False),     # K k = 64: two 32-row chunks of the real flush loop
    ("det", 192, 8, 16, False),    # 128
    ("det", 192, 8, 32, False),    # 256
    ("det", 96, 4, 16, True),      # complex, K k = 64: four 16-row chunks
    ("pf", 64, 2, 16, False),      # skew, 2 K k = 64
    ("pf", 96, 4, 12, False),      # skew, 96 columns
    ("pf", 48, 2, 16, True),       # skew complex, 64 columns: four chunks
    ("pf", 64, 8, 4, False),       # k = 8: 16 x 16 core, 64 columns
])
def test_flush_multichunk(kind, n, k, K, cplx):
    """The flush (Eq. 12 / Eq. 26) through MORE THAN ONE K-chunk of its staging loop in every
    instantiation (real / complex, det / skew), with every proposal applied so that the
    buffers fill to their full depth: K + 3 steps = one automatic full-depth flush plus the
    part-filled fold of get_inverse.  The flushed inverse is compared element by element."""
    st = _run(kind, 900 + n + K, 3, n, 2 * n, k, K, K + 3, cplx, forced=True,
              kernel={"flush": "flush_dmma_kernel"})
    assert st["max_inv_rel"] < max(1e-9, 50 * st["e_oracle"])


@pytest.mark.parametrize("n,k,K,kernel", [
    (512, 8, 32, "det_append_stream_real_kernel+det_append_finish_kernel"),   # even n: one DMMA stream for every k <= 8
    (1024, 8, 8, "det_append_stream_real_kernel+det_append_finish_kernel"),
    (300, 5, 5, "det_append_stream_real_kernel+det_append_finish_kernel"),    # ragged: n = 18.75 units, cap = 25 rows
    (512, 4, 8, "det_append_stream_real_kernel+det_append_finish_kernel"),    # k <= 4: 4 rows of N in shared memory
    (1024, 4, 32, "det_append_stream_real_kernel+det_append_finish_kernel"),
    (512, 2, 8, "det_append_stream_real_kernel+det_append_finish_kernel"),
    (1024, 1, 32, "det_append_stream_real_kernel+det_append_finish_kernel"),
    (130, 3, 7, "det_append_stream_real_kernel+det_append_finish_kernel"),    # n = 2 mod 16, cap = 21
    (301, 4, 4, "det_prep_kernel+det_append_kernel"),                         # odd n: rows not 16-byte aligned -> register-row pass
    (257, 8, 3, "det_prep_kernel+det_append_kernel"),                         # odd n, k = 8
])
def test_det_real_append_large_n(n, k, K, kernel):
    """Real-valued delayed append at the sizes of the configs[4] sweep, both variants; forced
    accept so that buffers fill and flush."""
    _run("det", 40 + n + k + K, 3, n, 2 * n, k, K, min(K, 10) + 3, walkers=[0, 2], scratch_every=1,
         forced=True, kernel={"append": kernel})


@pytest.mark.parametrize("n,k,K", [
    (1024, 4, 6),      # the configs[3] shape (k = 4), shallow buffer: flushes inside the run
    (1028, 3, 5),      # n a multiple of 4 but not of 16: part-filled last unit; cap = 15: part-filled buffer unit
    (1024, 1, 9),      # k = 1 through the 4-column fragments
])
def test_det_complex_append_stream(n, k, K):
    """Complex delayed append at n >= 1024: det_append_dmma_stream_kernel (rows of A0^-1 and of
    Abuf against N on the FP64 tensor pipe, no det_prep_kernel) + the in-place finish pass."""
    _run("det", 60 + n + k + K, 3, n, 2 * n, k, K, K + 4, cplx=True, walkers=[0, 2], scratch_every=1,
         forced=True, kernel={"append": "det_append_dmma_stream_kernel+det_append_finish_kernel"})


@pytest.mark.parametrize("n,k,K,cplx", [(128, 1, 4, False), (512, 2, 8, False), (512, 1, 4, False),
                                        (128, 2, 4, True), (64, 8, 0, False), (64, 8, 2, False)])
def test_pf_delayed_and_k8(n, k, K, cplx):
    """Pfaffian delayed kernels (pf_an / pf_y_colsum / pf_append / skew flush) above n = 50,
    and k = 8 (16 x 16 skew core), immediate and delayed."""
    _run("pf", 70 + n + k + K, 3, n, 2 * n, k, K, 20, cplx, walkers=[0, 2], scratch_every=1, forced=(k == 8))


@pytest.mark.parametrize("n,k,steps", [(128, 9, 6), (256, 16, 4), (256, 33, 3), (512, 64, 3), (200, 24, 3)])
def test_det_big_rank(n, k, steps):
    """Ranks 8 < k <= 64: ratio = gather + R = N C on the tensor
    pipe + Gauss-Jordan core, accept = row-dot pass + the k-column fold.  Every proposal applied
    (a Metropolis chain accepts almost no rank-16+ move on these inputs); n = 200: ragged tiles."""
    _run("det", 3000 + n + k, 3, n, 2 * n, k, 0, steps, forced=True,
         kernel={"ratio": "rowdot_dmma_kernel", "update": "flush_dmma_kernel"})


def test_det_big_rank_metropolis_and_mixed_ranks():
    """One handle with kmax = 16 serving a Metropolis chain of rank-12 moves: rejected walkers stay
    untouched, accepted ones follow the oracle."""
    _run("det", 3111, 8, 96, 192, 12, 0, 30, kmax=16, acc_range=(0.0, 1.0))


@pytest.mark.parametrize("kind,n,k,K", [("det", 64, 2, 0), ("det", 64, 2, 4), ("pf", 64, 1, 0), ("pf", 50, 2, 3)])
def test_forced_accept_chain(kind, n, k, K):
    """Forced-accept mode (what every ncu capture and the Fig. 2-style runs use) against the
    oracle with every proposal applied."""
    _run(kind, 300 + n + K, 4, n, 2 * n, k, K, 40, forced=True)


@pytest.mark.parametrize("kind,n,k,K", [("det", 64, 2, 0), ("det", 96, 4, 0), ("pf", 64, 1, 0), ("det", 64, 2, 8)])
def test_refresh_restores_bare_tolerance(kind, n, k, K):
    """lrux_*_refresh every 16 steps (<= 16 accepted updates between rebuilds): every ratio of
    a 400-step chain within the BARE 1e-10 of the from-scratch value, log-amplitude likewise --
    the accuracy guard does what it is for."""
    st = _run(kind, 77 + n + k, 6, n, 2 * n, k, K, 400, refresh_every=16, strict=True)
    assert st["pure_frac"] == 1.0


def test_det_config4_shape_reduced():
    """configs[3] shape reduced: complex128, k=4, delay K=32, n=256."""
    _run("det", wl.BASE_SEED + 4, 6, 256, 512, 4, 32, 80, cplx=True, walkers=[0, 5], scratch_every=5)


@pytest.mark.parametrize("kmax,K,cplx", [(8, 32, False), (8, 96, False), (8, 48, True)])
def test_large_delay_coefficient_staging(kmax, K, cplx):
    """Delay shapes whose ratio kernel stages > 40 KB of coefficients (opt-in dynamic shared
    memory): f64 kmax=8 K=96 (48 KB) and c128 kmax=8 K=48 used to pass init and then fail
    every ratio call; pf kmax=8 K=32 used to be rejected outright."""
    _run("det", 5 + K, 2, 64, 128, 2, K, 12, cplx, kmax=kmax)
    _run("pf", 6 + K, 2, 64, 128, 2, min(K, 32), 12, cplx, kmax=kmax)


@pytest.mark.parametrize("kind,n,k,K", [("det", 64, 2, 0), ("det", 96, 2, 4), ("pf", 64, 1, 0), ("pf", 200, 1, 0),
                                        ("det", 1024, 8, 0)])
def test_cuda_graph_replay_equals_stream_launches(kind, n, k, K):
    """mc.Chain.capture: one step captured into a CUDA graph (device-side step counter) and
    replayed gives, bit for bit, the chain that stream launches give -- ratios, decisions,
    inverse, amplitude.  Includes the cluster launches (pf n=200, det n=1024 k=8 at n <= 1024: no
    cluster; pf_cluster_k1) and the delayed path with its flush."""
    from paper_2602_05255_b200 import mc

    seed = 88 + n
    orb, occ, unocc = pu.make_inputs(kind, seed, 6, n, 2 * n)
    dev = "cuda"
    mk = lambda: mc.Chain(kind, torch.as_tensor(orb, device=dev), torch.as_tensor(occ, device=dev),
                          torch.as_tensor(unocc, device=dev), k=k, K=K, seed=seed)
    a, b = mk(), mk()
    T, pre = 24, 3
    ra, ma = [], []
    for t in range(T):
        a.step(t)
        ra.append(a.ratio.clone())
        ma.append(a.mask.clone())
    for t in range(pre):
        b.step(t)
    b.capture(pre)
    for t in range(pre, T):
        b.replay()
        assert torch.equal(b.ratio, ra[t]) and torch.equal(b.mask, ma[t]), t
    assert int(b.d_step[0].item()) == T and int(b.d_step[1].item()) == 0
    assert torch.equal(a.walkers.get_inverse(), b.walkers.get_inverse())
    assert torch.equal(a.occ, b.occ) and int(a.naccept.item()) == int(b.naccept.item())
    pa, la = a.walkers.get_amplitude()
    pb, lb = b.walkers.get_amplitude()
    assert torch.equal(pa, pb) and torch.equal(la, lb)
    assert b.launches_per_replay >= 5


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
