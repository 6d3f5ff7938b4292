"""Edge cases of the CUDA path against the oracle's plain definitions: degenerate sizes,
nothing accepted, variable k under one handle, a second ratio replacing the pending one,
explicit flush, get_inverse with a half-full delay buffer."""
import numpy as np
import pytest
import torch

from oracle import lrux_oracle as orc
from paper_2602_05255_b200 import lrux

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _t(x, dtype=None):
    return torch.as_tensor(np.ascontiguousarray(x), device=DEV, dtype=dtype)


def _replace_rows(A, idx, rows):
    B = A.copy()
    B[idx, :] = rows
    return B


@pytest.mark.parametrize("n,k", [(1, 1), (2, 2), (8, 8), (3, 1)])
def test_det_degenerate_sizes(n, k):
    """n = 1, k = n (every row replaced at once), odd n."""
    rng = np.random.default_rng(n * 10 + k)
    W = 3
    A = rng.standard_normal((W, n, n)) + 2 * np.eye(n)
    wk = lrux.DetWalkers(_t(A), kmax=k)
    idx = np.stack([rng.permutation(n)[:k] for _ in range(W)]).astype(np.int32)
    rows = rng.standard_normal((W, k, n))
    r = wk.ratio_(_t(idx), _t(rows)).cpu().numpy()
    wk.accept(torch.ones(W, dtype=torch.uint8, device=DEV))
    inv = wk.get_inverse().cpu().numpy()
    ph, la = wk.get_amplitude()
    for w in range(W):
        B = _replace_rows(A[w], idx[w], rows[w])
        assert r[w] == pytest.approx(orc.det(B) / orc.det(A[w]), rel=1e-10)
        assert np.abs(B @ inv[w] - np.eye(n)).max() < 1e-9
        sph, sla = orc.slogdet(B)
        assert la[w].item() == pytest.approx(sla, abs=1e-10 * max(1, abs(sla)))
        assert ph[w].item() == sph


@pytest.mark.parametrize("K", [0, 3])
def test_nothing_accepted_and_single_walker(K):
    """mask = 0 everywhere (empty work lists in every accept kernel), W = 1."""
    rng = np.random.default_rng(5)
    n, k = 20, 2
    A = rng.standard_normal((1, n, n))
    wk = lrux.DetWalkers(_t(A), kmax=k, K=K)
    before = wk.get_inverse().cpu().numpy()
    for _ in range(4):
        idx = rng.permutation(n)[:k].astype(np.int32)[None]
        wk.ratio_(_t(idx), _t(rng.standard_normal((1, k, n))))
        wk.accept(torch.zeros(1, dtype=torch.uint8, device=DEV))
    wk.flush()
    assert np.array_equal(wk.get_inverse().cpu().numpy(), before)
    assert wk.info.cpu().tolist() == [0]


def test_variable_k_second_ratio_and_explicit_flush():
    """One handle (kmax = 4, K = 3): proposals of k = 1, 4, 2, 3 rows; a second ratio
    before accept replaces the pending proposal; get_inverse folds a half-full buffer;
    every ratio and the final inverse against the oracle's plain definitions."""
    rng = np.random.default_rng(9)
    W, n, kmax = 4, 24, 4
    A = rng.standard_normal((W, n, n))
    cur = A.copy()
    wk = lrux.DetWalkers(_t(A), kmax=kmax, K=3)
    logabs = np.array([orc.slogdet(A[w])[1] for w in range(W)])
    for step, k in enumerate([1, 4, 2, 3, 1, 2]):
        # a throw-away proposal first: must leave no trace
        idx0 = np.stack([rng.permutation(n)[:k] for _ in range(W)]).astype(np.int32)
        wk.ratio_(_t(idx0), _t(rng.standard_normal((W, k, n))))
        idx = np.stack([rng.permutation(n)[:k] for _ in range(W)]).astype(np.int32)
        rows = rng.standard_normal((W, k, n))
        r = wk.ratio_(_t(idx), _t(rows)).cpu().numpy()
        mask = (rng.random(W) < 0.7).astype(np.uint8)
        wk.accept(_t(mask))
        for w in range(W):
            B = _replace_rows(cur[w], idx[w], rows[w])
            assert r[w] == pytest.approx(orc.det(B) / orc.det(cur[w]), rel=1e-9)
            if mask[w]:
                cur[w] = B
                logabs[w] += np.log(abs(r[w]))
        if step == 3:
            wk.flush()                      # explicit flush in the middle
    inv = wk.get_inverse().cpu().numpy()     # implies flush of whatever is buffered
    _, la = wk.get_amplitude()
    for w in range(W):
        assert np.abs(cur[w] @ inv[w] - np.eye(n)).max() < 1e-9
        assert la[w].item() == pytest.approx(orc.slogdet(cur[w])[1], abs=1e-9)
    assert not wk.info.cpu().numpy().any()


def test_pf_degenerate_and_k_equals_half_n():
    """Pfaffian: n = 2 (k = 1 replaces the only pair), n = 8 with k = 4."""
    rng = np.random.default_rng(21)
    for n, k in ((2, 1), (8, 4), (6, 2)):
        W, M = 3, 2 * n + 2
        g = rng.standard_normal((W, M, M))
        F = np.triu(g, 1) - np.triu(g, 1).transpose(0, 2, 1)
        occ = np.stack([rng.permutation(M)[:n] for _ in range(W)])
        A = np.stack([F[w][np.ix_(occ[w], occ[w])] for w in range(W)])
        wk = lrux.PfWalkers(_t(A), kmax=k)
        idx = np.stack([rng.permutation(n)[:k] for _ in range(W)]).astype(np.int32)
        newocc = occ.copy()
        for w in range(W):
            free = [o for o in range(M) if o not in occ[w]]
            newocc[w, idx[w]] = rng.permutation(free)[:k]
        B = np.stack([F[w][np.ix_(newocc[w], newocc[w])] for w in range(W)])
        rows = np.stack([B[w][idx[w], :] for w in range(W)])
        r = wk.ratio_(_t(idx), _t(rows)).cpu().numpy()
        wk.accept(torch.ones(W, dtype=torch.uint8, device=DEV))
        inv = wk.get_inverse().cpu().numpy()
        for w in range(W):
            assert r[w] == pytest.approx(orc.pf(B[w]) / orc.pf(A[w]), rel=1e-9)
            assert np.abs(B[w] @ inv[w] - np.eye(n)).max() < 1e-8
            assert np.array_equal(inv[w], -inv[w].T)


def test_delay_depth_limit_is_reported():
    """K*kmax*kt*sizeof(elem) > 160 KiB of staged coefficients: rejected at init, not at the
    first ratio call."""
    with pytest.raises(lrux.LruxError) as e:
        lrux.DetWalkers(torch.eye(16, dtype=torch.complex128, device=DEV)[None], kmax=8, K=200)
    assert e.value.status == lrux.EUNSUPPORTED
    lrux.DetWalkers(torch.eye(16, dtype=torch.complex128, device=DEV)[None], kmax=8, K=64)   # 64 KiB: fine


@pytest.mark.parametrize("kind,dtype,K", [("det", np.float64, 0), ("det", np.complex128, 3), ("pf", np.float64, 0),
                                          ("pf", np.float64, 2)])
def test_refresh_rebuilds_inverse_and_amplitude(kind, dtype, K):
    """lrux_*_refresh: after a run of accepted updates — with factors still
    unflushed when K > 0 — a refresh from the walkers' current matrices gives the from-scratch
    inverse and amplitude of the oracle, drops the delay factors, and the chain goes on."""
    rng = np.random.default_rng(77 + K)
    W, n, k = 3, 24, 2
    cplx = dtype == np.complex128

    def rnd(*shape):
        x = rng.standard_normal(shape)
        return x + 1j * rng.standard_normal(shape) if cplx else x

    def skew(x):
        return np.triu(x, 1) - np.triu(x, 1).transpose(0, 2, 1)

    A = skew(rnd(W, n, n)) if kind == "pf" else rnd(W, n, n) + 3 * np.eye(n)
    wk = (lrux.PfWalkers if kind == "pf" else lrux.DetWalkers)(_t(A), kmax=k, K=K)
    ones = torch.ones(W, dtype=torch.uint8, device=DEV)

    def step(A):
        idx = np.stack([rng.permutation(n)[:k] for _ in range(W)]).astype(np.int32)
        B = A.copy()
        rows = np.empty((W, k, n), dtype=A.dtype)
        for w in range(W):
            new = rnd(k, n)
            if kind == "pf":
                for a, p in enumerate(idx[w]):
                    new[a, p] = 0.0
                for a, p in enumerate(idx[w]):          # crossing entries stay skew
                    for b, q in enumerate(idx[w]):
                        if b > a:
                            new[b, p] = -new[a, q]
                for a, p in enumerate(idx[w]):
                    B[w, p, :] = new[a]
                    B[w, :, p] = -new[a]
            else:
                B[w, idx[w], :] = new
            rows[w] = new
        r = wk.ratio_(_t(idx), _t(rows)).cpu().numpy()
        wk.accept(ones)
        return B, r

    amp = orc.slogpf if kind == "pf" else orc.slogdet
    for _ in range(5):        # K = 3 / 2: the buffers are partly filled when the refresh comes
        A, _ = step(A)
    # poison the tracked state's accuracy claim: refresh must not depend on it
    wk.refresh(_t(A))
    inv = wk.get_inverse().cpu().numpy()
    ph, la = wk.get_amplitude()
    assert wk.info.cpu().numpy().tolist() == [0] * W
    for w in range(W):
        assert np.abs(A[w] @ inv[w] - np.eye(n)).max() < 1e-11
        p0, l0 = amp(A[w])
        assert la[w].item() == pytest.approx(l0, abs=1e-11)
        assert abs(complex(ph[w].item()) - complex(p0)) < 1e-11
        if kind == "pf":
            assert np.array_equal(inv[w], -inv[w].T)
    A_old = A
    A, r = step(A)            # the chain continues from the refreshed state
    for w in range(W):
        p1, l1 = amp(A[w])
        p0, l0 = amp(A_old[w])
        assert r[w] == pytest.approx(complex(p1) / complex(p0) * np.exp(l1 - l0), rel=1e-9)
    # a refresh from a singular matrix raises bit 1 for that walker only
    S = A.copy()
    S[1] = 0.0
    wk.refresh(_t(S))
    torch.cuda.synchronize()
    assert wk.info.cpu().numpy().tolist() == [0, 1, 0]
    wk.refresh(_t(A))         # and a good one clears it again
    inv = wk.get_inverse().cpu().numpy()
    assert wk.info.cpu().numpy().tolist() == [0] * W
    assert np.abs(A[1] @ inv[1] - np.eye(n)).max() < 1e-11


_GUARD_SHAPES = [
    # kind, n, k, K, cplx, forced : one per kernel family the dispatcher can pick
    ("det", 33, 1, 0, False, False), ("det", 64, 2, 4, False, False), ("det", 96, 4, 8, True, False),
    ("det", 130, 8, 0, False, True), ("det", 128, 8, 4, False, True), ("det", 256, 3, 0, False, True),
    ("det", 192, 4, 0, True, True), ("det", 512, 1, 16, False, False), ("det", 1026, 4, 0, False, True),
    ("det", 128, 16, 0, False, True), ("det", 64, 5, 3, False, True), ("det", 47, 2, 5, True, True),
    ("pf", 32, 1, 0, False, False), ("pf", 64, 2, 4, False, True), ("pf", 130, 1, 8, False, False),
    ("pf", 96, 4, 0, False, True),
    # kernels added late in round 2
    ("det", 1028, 3, 5, True, True),      # det_append_dmma_stream_kernel + in-place finish (ragged units)
    ("det", 516, 4, 6, False, True),      # det_append_stream_real_kernel, shared copy of N
    ("det", 100, 3, 4, False, True),      # ... per-warp copies of N; det_ratio_kernel with a delay buffer
    ("det", 72, 4, 0, False, True),       # det_update_dmma_warp_kernel, det_ratio_warp_kernel
    ("det", 250, 8, 0, False, True),      # 32 blocks per warp, DMMA partial R in the ratio
    ("pf", 100, 3, 0, False, True),       # pf_update_dmma_warp_kernel, row-dot Y pass
    ("pf", 1040, 2, 0, False, True),      # pf_update_dmma_kernel with column ranges
]


@pytest.mark.parametrize("kind,n,k,K,cplx,forced", _GUARD_SHAPES)
def test_no_write_outside_the_state_buffer(kind, n, k, K, cplx, forced):
    """Stand-in for compute-sanitizer (closed on this pool, profiles/r02_sanitizer.md): 4 KiB of
    guard bytes on both sides of the state buffer stay intact over a chain that fills and
    flushes the delay buffer, and two runs from the same inputs are bit-identical (a race or a
    read of uninitialised memory would show up as a difference)."""
    import parity_util as pu
    from paper_2602_05255_b200 import mc

    W, M, seed, steps = 5, 2 * n, 77 + n, 3 * max(K, 1) + 6
    orb, occ, unocc = pu.make_inputs(kind, seed, W, n, M, cplx)
    out = []
    for _ in range(2):
        ch = mc.Chain(kind, _t(orb), _t(occ), _t(unocc), k=k, K=K, seed=seed, guard=4096)
        ratios = []
        for t in range(steps):
            ch.step(t, forced)
            ratios.append(ch.ratio.clone())
        inv = ch.walkers.get_inverse()
        ph, la = ch.walkers.get_amplitude()
        torch.cuda.synchronize()
        assert ch.walkers.guards_intact()
        out.append((torch.stack(ratios).cpu(), inv.cpu(), ph.cpu(), la.cpu(), ch.occ.cpu()))
    for a, b in zip(*out):
        assert torch.equal(torch.view_as_real(a) if a.is_complex() else a,
                           torch.view_as_real(b) if b.is_complex() else b)
