"""General update factors (Eq. 6-9, and the dense form of
Eq. 2-5): lrux_det_ratio_general / lrux_det_accept against the oracle's det_lru driven with the
same factors written out densely, and against the determinant recomputed from scratch."""
import numpy as np
import pytest
import torch

from oracle import c_oracle as orc
from paper_2602_05255_b200 import lrux

pytestmark = pytest.mark.gpu
DEV = "cuda"


def _t(x, dtype=None):
    return torch.as_tensor(np.ascontiguousarray(x), device=DEV, dtype=dtype)


def _rand(rng, shape, cplx):
    x = rng.standard_normal(shape)
    return x + 1j * rng.standard_normal(shape) if cplx else x


def _factor(rng, W, n, kd, ke, cplx, scale):
    """kd dense columns + ke distinct one-hot columns; returns (dense [W][kd][n] or None,
    idx [W][ke] or None, the factor written out densely [W][n][kd+ke])."""
    dense = _rand(rng, (W, kd, n), cplx) * scale if kd else None
    idx = np.stack([rng.permutation(n)[:ke] for _ in range(W)]).astype(np.int32) if ke else None
    full = np.zeros((W, n, kd + ke), np.complex128 if cplx else np.float64)
    for w in range(W):
        for a in range(kd):
            full[w, :, a] = dense[w, a]
        for a in range(ke):
            full[w, idx[w, a], kd + a] = 1.0
    return dense, idx, full


CASES = [
    # name, (u_kd, u_ke), (v_kd, v_ke)
    ("row replacement, Eq. 6/8", (1, 0), (0, 1)),
    ("row replacement k=3", (3, 0), (0, 3)),
    ("column replacement, Eq. 7", (0, 1), (1, 0)),
    ("column replacement k=2", (0, 2), (2, 0)),
    ("row + column, Eq. 9", (1, 1), (1, 1)),
    ("row + column k=2+2", (2, 2), (2, 2)),
    ("dense rank 1, Eq. 2-5", (1, 0), (1, 0)),
    ("dense rank 5", (5, 0), (5, 0)),
    ("dense rank 8", (8, 0), (8, 0)),
    ("mixed 3 dense + 1 one-hot / 1 dense + 3 one-hot", (3, 1), (1, 3)),
]


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("name,uf,vf", CASES)
@pytest.mark.parametrize("n,K", [(48, 0), (130, 3)])
def test_general_factors_follow_the_oracle(name, uf, vf, n, K, cplx):
    import zlib

    rng = np.random.default_rng(zlib.crc32(("%s %d %d" % (name, n, cplx)).encode()))
    W, k, steps = 5, uf[0] + uf[1], 6
    A = _rand(rng, (W, n, n), cplx) / np.sqrt(n)
    wk = lrux.DetWalkers(_t(A), kmax=k, K=K)
    Ainv = np.stack([orc.inv(A[w]) for w in range(W)])       # the oracle's tracked inverse
    ph0, la0 = wk.get_amplitude()
    logabs = la0.cpu().numpy().copy()
    if K:   # put something into the delay buffers first: the general call must fold it
        idx = np.stack([rng.permutation(n)[:1] for _ in range(W)]).astype(np.int32)
        rows = _rand(rng, (W, 1, n), cplx) / np.sqrt(n)
        r0 = wk.ratio_(_t(idx), _t(rows)).cpu().numpy().copy()
        wk.accept(torch.ones(W, dtype=torch.uint8, device=DEV))
        for w in range(W):
            u = (rows[w, 0] - A[w, idx[w, 0]])[:, None]
            v = np.zeros((n, 1), A.dtype)
            v[idx[w, 0], 0] = 1
            r, Ainv[w] = orc.det_lru(Ainv[w], u, v, True)
            assert abs(r0[w] - r) <= 1e-9 * abs(r)
            A[w, idx[w, 0]] = rows[w, 0]
            logabs[w] += np.log(abs(r))
    worst = 0.0
    for t in range(steps):
        ud, ui, U = _factor(rng, W, n, uf[0], uf[1], cplx, 0.3 / np.sqrt(n))
        # sizes: v u^T ~ 0.3 |A_ij| for dense x dense; a pure column replacement (u one-hot) gets
        # deltas of that size directly
        vd, vi, V = _factor(rng, W, n, vf[0], vf[1], cplx, 1.0 if uf[0] else 0.3 / np.sqrt(n))
        r_gpu = wk.ratio_general_(None if ud is None else _t(ud), None if ui is None else _t(ui),
                                  None if vd is None else _t(vd), None if vi is None else _t(vi)).cpu().numpy().copy()
        mask = (rng.random(W) < 0.7).astype(np.uint8)
        wk.accept(_t(mask))
        for w in range(W):
            A1 = A[w] + V[w] @ U[w].T
            r_lemma, new = orc.det_lru(Ainv[w], U[w], V[w], True)          # Eq. 3-5 with dense factors
            (p1, l1), (p0, l0) = orc.slogdet(A1), orc.slogdet(A[w])
            r_scratch = (p1 / p0) * np.exp(l1 - l0)
            e_orc = abs(r_lemma - r_scratch) / abs(r_scratch)
            rel = abs(r_gpu[w] - r_scratch) / abs(r_scratch)
            worst = max(worst, rel)
            assert rel <= min(1e-10 + 4 * e_orc, 1e-8), (name, t, w, r_gpu[w], r_scratch, r_lemma)
            if mask[w]:
                A[w], Ainv[w] = A1, new
                logabs[w] += np.log(abs(r_scratch))
    assert not wk.info.cpu().numpy().any()
    inv = wk.get_inverse().cpu().numpy()
    ph, la = wk.get_amplitude()
    for w in range(W):
        assert np.abs(A[w] @ inv[w] - np.eye(n)).max() < 1e-9
        assert np.abs(inv[w] - Ainv[w]).max() <= 1e-9 * np.abs(Ainv[w]).max()
        assert abs(la[w].item() - logabs[w]) < 1e-9
    assert "gen_core_kernel" in wk.kernel_name(lrux.PROF_RATIO)
    assert "flush_dmma_kernel" in wk.kernel_name(lrux.PROF_UPDATE)
    print("general[%s n=%d %s]: worst relative ratio error %.2e" % (name, n, "c128" if cplx else "f64", worst))


def test_general_factors_argument_checks_and_bad_index():
    W, n = 3, 16
    rng = np.random.default_rng(5)
    wk = lrux.DetWalkers(_t(rng.standard_normal((W, n, n))), kmax=2, K=0)
    x = _t(rng.standard_normal((W, 1, n)))
    good = _t(np.array([[1], [2], [3]], np.int32))
    with pytest.raises(ValueError):                       # column counts differ
        wk.ratio_general_(x, good, x, None)
    with pytest.raises(lrux.LruxError) as e:              # k > kmax
        wk.ratio_general_(_t(rng.standard_normal((W, 3, n))), None, None, _t(np.zeros((W, 3), np.int32)))
    assert e.value.status == lrux.EINVAL
    bad = _t(np.array([[1], [99], [3]], np.int32))
    r = wk.ratio_general_(x, None, None, bad).cpu().numpy()
    assert np.isfinite(r[0]) and np.isnan(r[1]) and np.isfinite(r[2])
    before = wk.get_inverse().cpu().numpy()
    wk.ratio_general_(x, None, None, bad)
    wk.accept(torch.ones(W, dtype=torch.uint8, device=DEV))
    after = wk.get_inverse().cpu().numpy()
    assert (wk.info.cpu().numpy()[1] & 2) and np.array_equal(before[1], after[1])
    assert not np.array_equal(before[0], after[0])
