"""lrux_det_ratio_noalloc (include/lrux.h): the allocation-free determinant ratio against the
existing handle path (lrux_det_ratio), on calls in a row that share the library's fixed scratch
array.  Collected last on purpose (the run uses -x)."""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2602_05255_b200 import lrux

RTOL, ATOL = 1e-10, 1e-12      # the bare parity tolerance of DESIGN.md reading 14


def _problem(seed, W, n, k, cplx):
    rng = np.random.default_rng(seed)
    g = (lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)) if cplx else (lambda *s: rng.standard_normal(s))
    A = g(W, n, n) / np.sqrt(n) + np.eye(n)
    idx = np.stack([rng.permutation(n)[:k] for _ in range(W)]).astype(np.int32)
    rows = g(W, k, n) / np.sqrt(n)
    rows[np.arange(W)[:, None], np.arange(k)[None, :], idx] += 1.0
    dev = "cuda"
    return (torch.as_tensor(A, device=dev), torch.as_tensor(idx, device=dev), torch.as_tensor(rows, device=dev))


def _existing_path(A, idx, rows):
    """Ratio through a handle (state buffer allocated by the caller) and the stored A^-T."""
    wk = lrux.DetWalkers(A, kmax=int(idx.shape[1]))
    Ti = wk.get_inverse().transpose(1, 2).contiguous()
    ref = wk.ratio_(idx, rows).clone()
    torch.cuda.synchronize()
    assert wk.info.cpu().numpy().max() == 0
    return Ti, ref


def _close(a, b):
    return torch.allclose(a, b, rtol=RTOL, atol=ATOL)


@pytest.mark.gpu
def test_noalloc_ratio_matches_handle_path_on_calls_in_a_row():
    cases = [(11, 900, 96, 8, False),      # 900*64*8 B = 450 KiB of the 1 MiB scratch
             (12, 300, 65, 3, True),       # complex, smaller: runs over the first call's leftovers
             (13, 2048, 40, 1, False),
             (14, 257, 130, 5, False)]
    prepared = []
    for seed, W, n, k, cplx in cases:
        A, idx, rows = _problem(seed, W, n, k, cplx)
        Ti, ref = _existing_path(A, idx, rows)
        prepared.append((Ti, idx, rows, ref, torch.empty_like(ref)))
    torch.cuda.synchronize()
    # number of allocation EVENTS of torch's caching allocator (monotonic: frees by the garbage
    # collector of earlier tests' tensors do not move it)
    before = torch.cuda.memory_stats()["allocation.all.allocated"]
    for Ti, idx, rows, ref, out in prepared:            # back to back on one stream, no sync between
        lrux.det_ratio_noalloc(Ti, idx, rows, out)
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == before   # the binding allocated nothing either
    torch.cuda.synchronize()
    for Ti, idx, rows, ref, out in prepared:
        assert torch.isfinite(torch.view_as_real(out) if out.is_complex() else out).all()
        assert _close(out, ref), (out - ref).abs().max().item()
    # the same inputs again, after other problems have used the scratch: bit-identical
    Ti, idx, rows, ref, out = prepared[0]
    again = torch.empty_like(out)
    lrux.det_ratio_noalloc(Ti, idx, rows, again)
    torch.cuda.synchronize()
    assert torch.equal(again, out)


@pytest.mark.gpu
def test_noalloc_bad_indices_and_limit():
    A, idx, rows = _problem(21, 64, 32, 2, False)
    Ti, ref = _existing_path(A, idx, rows)
    idx = idx.clone()
    idx[3, 1] = idx[3, 0]          # duplicate
    idx[5, 0] = 32                 # out of range
    out = torch.empty_like(ref)
    lrux.det_ratio_noalloc(Ti, idx, rows, out)
    torch.cuda.synchronize()
    bad = torch.zeros(64, dtype=torch.bool, device="cuda")
    bad[3] = bad[5] = True
    assert torch.isnan(out[bad]).all()
    assert _close(out[~bad], ref[~bad])
    # one element past the fixed scratch: rejected on the host, output untouched
    W, k = lrux.NOALLOC_SCRATCH_BYTES // (8 * 4) + 1, 2
    big_idx = torch.zeros((W, k), dtype=torch.int32, device="cuda")
    big_idx[:, 1] = 1
    big_rows = torch.zeros((W, k, 2), dtype=torch.float64, device="cuda")
    big_Ti = torch.zeros((W, 2, 2), dtype=torch.float64, device="cuda")
    big_out = torch.full((W,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(lrux.LruxError) as e:
        lrux.det_ratio_noalloc(big_Ti, big_idx, big_rows, big_out)
    assert e.value.status == lrux.ELIMIT and "LRUX_NOALLOC_SCRATCH_BYTES" in str(e.value)
    torch.cuda.synchronize()
    assert (big_out == 7.0).all()
    lrux.det_ratio_noalloc(big_Ti[:-1], big_idx[:-1], big_rows[:-1], big_out[:-1])   # exactly at the limit: accepted
    torch.cuda.synchronize()
    assert (big_out[:-1] == 0.0).all()


def test_noalloc_limit_is_checked_before_any_cuda_call():
    """Host-side argument checks (no GPU): null pointers, rank and the scratch limit."""
    lib = lrux.load_library()
    p = C.c_void_p(256)            # never dereferenced: every call below returns before a launch
    f = lib.lrux_det_ratio_noalloc
    assert f(4, 8, 1, lrux.F64, None, p, p, p, None) == lrux.EINVAL
    assert f(4, 8, 9, lrux.F64, p, p, p, p, None) == lrux.EINVAL
    assert f(0, 8, 1, lrux.F64, p, p, p, p, None) == lrux.EINVAL
    assert f(4, 8, 1, 5, p, p, p, p, None) == lrux.EINVAL
    assert f(2049, 64, 8, lrux.F64, p, p, p, p, None) == lrux.ELIMIT        # 2049*64*8 B > 1 MiB
    assert f(1025, 64, 8, lrux.C128, p, p, p, p, None) == lrux.ELIMIT
    assert f(1 << 40, 64, 1, lrux.F64, p, p, p, p, None) == lrux.ELIMIT
    assert b"LRUX_ELIMIT" in lib.lrux_status_string(lrux.ELIMIT)
