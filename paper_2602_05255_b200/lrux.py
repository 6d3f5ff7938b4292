"""Thin ctypes binding of include/lrux.h and include/lrux_harness.h.

Argument marshalling only: every step of the path runs in the CUDA kernels of
lib/liblrux.so.  torch is used for device memory and streams.  There is no CPU
fallback: a missing library raises at import of the symbols.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "lib", "liblrux.so")

F64, C128 = 0, 1
OK, EINVAL, ESTATE, EWORKSPACE, EUNSUPPORTED, ECUDA, ELIMIT = range(7)
NOALLOC_SCRATCH_BYTES = 1 << 20
MAX_K = 64
PROF_RATIO, PROF_UPDATE, PROF_APPEND, PROF_FLUSH, PROF_YPASS = range(5)

_vp, _i32, _i64, _u64, _sz = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_size_t

# name -> argtypes; restype is int (lrux_status_t) unless listed in _RESTYPE
SIGNATURES = {
    "lrux_det_state_bytes": [_i64, _i32, _i32, _i32, C.c_int, C.POINTER(_sz)],
    "lrux_pf_state_bytes": [_i64, _i32, _i32, _i32, C.c_int, C.POINTER(_sz)],
    "lrux_det_init": [C.POINTER(_vp), _i64, _i32, _i32, _i32, C.c_int, _vp, _vp, _sz, _vp, _vp],
    "lrux_pf_init": [C.POINTER(_vp), _i64, _i32, _i32, _i32, C.c_int, _vp, _vp, _sz, _vp, _vp],
    "lrux_det_attach": [C.POINTER(_vp), _i64, _i32, _i32, _i32, C.c_int, _vp, _sz, _vp],
    "lrux_pf_attach": [C.POINTER(_vp), _i64, _i32, _i32, _i32, C.c_int, _vp, _sz, _vp],
    "lrux_det_refresh": [_vp, _vp, _vp],
    "lrux_pf_refresh": [_vp, _vp, _vp],
    "lrux_det_ratio": [_vp, _i32, _vp, _vp, _vp, _vp],
    "lrux_pf_ratio": [_vp, _i32, _vp, _vp, _vp, _vp],
    "lrux_det_ratio_general": [_vp, _i32, _i32, _vp, _vp, _i32, _vp, _vp, _vp, _vp],
    "lrux_det_ratio_noalloc": [_i64, _i32, _i32, C.c_int, _vp, _vp, _vp, _vp, _vp],
    "lrux_det_accept": [_vp, _vp, _vp],
    "lrux_pf_accept": [_vp, _vp, _vp],
    "lrux_det_flush": [_vp, _vp],
    "lrux_pf_flush": [_vp, _vp],
    "lrux_det_get_amplitude": [_vp, _vp, _vp, _vp],
    "lrux_pf_get_amplitude": [_vp, _vp, _vp, _vp],
    "lrux_det_get_inverse": [_vp, _vp, _vp],
    "lrux_pf_get_inverse": [_vp, _vp, _vp],
    "lrux_get_flush_count": [_vp, _vp, _vp],
    "lrux_launch_count": [_vp, C.POINTER(_i64)],
    "lrux_kernel_name": [_vp, _i32],
    "lrux_profile_enable": [_vp, _i32],
    "lrux_profile_read": [_vp, _i32, C.POINTER(C.c_double), C.POINTER(_i64)],
    "lrux_destroy": [_vp],
    "lrux_status_string": [C.c_int],
    "lruxh_det_propose": [_u64, _i64, _i64, _i64, _i32, _i32, _i32, C.c_int, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp],
    "lruxh_pf_propose": [_u64, _i64, _i64, _i64, _i32, _i32, _i32, C.c_int, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp],
    "lruxh_decide": [_u64, _i64, _i64, _i64, _i32, _i32, _i32, C.c_int, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp],
}
_RESTYPE = {"lrux_status_string": C.c_char_p, "lrux_kernel_name": C.c_char_p}

_lib = None


def load_library():
    """dlopen lib/liblrux.so and declare every symbol of the two headers."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                "liblrux.so is not built: run `python -m paper_2602_05255_b200.build` "
                "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        for name, argtypes in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.argtypes = argtypes
            fn.restype = _RESTYPE.get(name, C.c_int)
        _lib = lib
    return _lib


class LruxError(RuntimeError):
    def __init__(self, status):
        self.status = status
        super().__init__(load_library().lrux_status_string(status).decode())


def _check(status):
    if status != OK:
        raise LruxError(status)


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _ptr(t):
    return C.c_void_p(t.data_ptr())


def _dt(dtype):
    if dtype == torch.float64:
        return F64
    if dtype == torch.complex128:
        return C128
    raise TypeError("lrux supports float64 and complex128 only")


def state_bytes(kind, W, n, kmax, K, dtype):
    out = _sz(0)
    fn = getattr(load_library(), "lrux_%s_state_bytes" % kind)
    _check(fn(W, n, kmax, K, _dt(dtype), C.byref(out)))
    return out.value


class _Walkers:
    """Owner of one lrux handle plus the caller-side buffers it points into."""

    kind = "det"

    def __init__(self, A0, kmax=1, K=0, stream=None, guard=0):
        """``guard`` > 0 (tests): that many bytes of 0xA5 before and after the state buffer,
        checked by ``guards_intact()`` -- an out-of-bounds write detector that needs no tool."""
        lib = load_library()
        if not A0.is_cuda:
            raise ValueError("A0 must be a CUDA tensor (no CPU path)")
        A0 = A0.contiguous()
        self.W, self.n = int(A0.shape[0]), int(A0.shape[1])
        self.kmax, self.K, self.dtype, self.device = int(kmax), int(K), A0.dtype, A0.device
        nbytes = state_bytes(self.kind, self.W, self.n, self.kmax, self.K, self.dtype)
        self._guard = g = (int(guard) + 255) // 256 * 256
        self.state = torch.empty(nbytes + 256 + 2 * g, dtype=torch.uint8, device=self.device)
        off = (-self.state.data_ptr()) % 256 + g
        self._state_ptr = self.state.data_ptr() + off
        self._nbytes = nbytes
        if g:
            self.state[:off].fill_(0xA5)
            self.state[off + nbytes:].fill_(0xA5)
        self.info = torch.zeros(self.W, dtype=torch.int32, device=self.device)
        self.ratio = torch.empty(self.W, dtype=self.dtype, device=self.device)
        self._h = C.c_void_p()
        fn = getattr(lib, "lrux_%s_init" % self.kind)
        _check(fn(C.byref(self._h), self.W, self.n, self.kmax, self.K, _dt(self.dtype), _ptr(A0),
                  C.c_void_p(self._state_ptr), nbytes, _ptr(self.info), _stream(stream)))
        self._lib = lib

    def clone(self):
        """Independent copy of these walkers: byte copy of the state buffer + lrux_*_attach
        (no re-initialisation).  No proposal may be pending."""
        new = object.__new__(type(self))
        new._guard, new._nbytes = 0, getattr(self, "_nbytes", 0)
        for a in ("W", "n", "kmax", "K", "dtype", "device", "_lib"):
            setattr(new, a, getattr(self, a))
        nbytes = state_bytes(self.kind, self.W, self.n, self.kmax, self.K, self.dtype)
        new.state = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        off = (-new.state.data_ptr()) % 256
        new._state_ptr = new.state.data_ptr() + off
        src_off = self._state_ptr - self.state.data_ptr()
        new.state[off:off + nbytes].copy_(self.state[src_off:src_off + nbytes])
        new.info = self.info.clone()
        new.ratio = torch.empty(self.W, dtype=self.dtype, device=self.device)
        new._h = C.c_void_p()
        fn = getattr(self._lib, "lrux_%s_attach" % self.kind)
        _check(fn(C.byref(new._h), self.W, self.n, self.kmax, self.K, _dt(self.dtype),
                  C.c_void_p(new._state_ptr), nbytes, _ptr(new.info)))
        return new

    def _fn(self, name):
        return getattr(self._lib, "lrux_%s_%s" % (self.kind, name))

    def guards_intact(self):
        """True when no byte of the guard zones around the state buffer has changed
        (``guard=`` at construction); synchronises."""
        if not self._guard:
            return True
        off = self._state_ptr - self.state.data_ptr()
        lo, hi = self.state[:off], self.state[off + self._nbytes:]
        return bool((lo == 0xA5).all().item()) and bool((hi == 0xA5).all().item())

    def ratio_(self, idx, rows, out=None, stream=None):
        """lrux_*_ratio: idx int32 [W][k], rows [W][k][n]; returns ratio [W]."""
        k = int(idx.shape[1])
        out = self.ratio if out is None else out
        _check(self._fn("ratio")(self._h, k, _ptr(idx), _ptr(rows), _ptr(out), _stream(stream)))
        return out

    def ratio_general_(self, u_dense, u_idx, v_dense, v_idx, out=None, stream=None):
        """lrux_det_ratio_general: A' = A + v u^T, each factor = dense columns ([W][kd][n], or
        None) followed by one-hot columns (int32 [W][ke], or None).  Returns ratio [W]."""
        def split(dense, idx):
            kd = 0 if dense is None else int(dense.shape[1])
            ke = 0 if idx is None else int(idx.shape[1])
            return kd, ke, (None if dense is None else _ptr(dense.contiguous())), (None if idx is None else _ptr(idx.contiguous()))
        ukd, uke, ud, ui = split(u_dense, u_idx)
        vkd, vke, vd, vi = split(v_dense, v_idx)
        if ukd + uke != vkd + vke:
            raise ValueError("u and v must have the same number of columns")
        out = self.ratio if out is None else out
        _check(self._lib.lrux_det_ratio_general(self._h, ukd + uke, ukd, ud, ui, vkd, vd, vi, _ptr(out),
                                                _stream(stream)))
        return out

    def accept(self, mask, stream=None):
        """lrux_*_accept: mask uint8 [W]."""
        _check(self._fn("accept")(self._h, _ptr(mask), _stream(stream)))

    def flush(self, stream=None):
        _check(self._fn("flush")(self._h, _stream(stream)))

    def refresh(self, A, stream=None):
        """lrux_*_refresh: rebuild A^-1 and the amplitude from the walkers' current matrices
        A [W][n][n] (the library stores none)."""
        if not A.is_cuda or tuple(A.shape) != (self.W, self.n, self.n) or A.dtype != self.dtype:
            raise ValueError("A must be a CUDA tensor [W][n][n] of the walkers' dtype")
        A = A.contiguous()
        _check(self._fn("refresh")(self._h, _ptr(A), _stream(stream)))

    def get_amplitude(self, stream=None):
        phase = torch.empty(self.W, dtype=self.dtype, device=self.device)
        logabs = torch.empty(self.W, dtype=torch.float64, device=self.device)
        _check(self._fn("get_amplitude")(self._h, _ptr(phase), _ptr(logabs), _stream(stream)))
        return phase, logabs

    def get_inverse(self, stream=None):
        out = torch.empty((self.W, self.n, self.n), dtype=self.dtype, device=self.device)
        _check(self._fn("get_inverse")(self._h, _ptr(out), _stream(stream)))
        return out

    def flush_count(self, stream=None):
        """(walker flushes, buffer columns folded) since init; synchronises."""
        out = torch.zeros(2, dtype=torch.int64, device=self.device)
        _check(self._lib.lrux_get_flush_count(self._h, _ptr(out), _stream(stream)))
        return tuple(int(x) for x in out.cpu())

    def launch_count(self):
        c = _i64(0)
        _check(self._lib.lrux_launch_count(self._h, C.byref(c)))
        return c.value

    def kernel_name(self, cls):
        """Kernel most recently enqueued for class ``cls`` (PROF_*); "" when none."""
        return self._lib.lrux_kernel_name(self._h, cls).decode()

    def profile_enable(self, on=True):
        _check(self._lib.lrux_profile_enable(self._h, 1 if on else 0))

    def profile_read(self, cls):
        """(milliseconds, launches) of kernel class ``cls`` (PROF_*); synchronises."""
        ms, cnt = C.c_double(0.0), _i64(0)
        _check(self._lib.lrux_profile_read(self._h, cls, C.byref(ms), C.byref(cnt)))
        return ms.value, cnt.value

    def close(self):
        if self._h:
            self._lib.lrux_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class DetWalkers(_Walkers):
    """lrux_det_* on W walkers: A0 is [W][n][n] float64/complex128 on the GPU."""
    kind = "det"


class PfWalkers(_Walkers):
    """lrux_pf_* on W walkers: A0 is [W][n][n] skew-symmetric, n even."""
    kind = "pf"


# ---------------------------------------------------------------- harness
def det_ratio_noalloc(Ti, idx, rows, out, stream=None):
    """lrux_det_ratio_noalloc: r_w = det(N_w A_w^-1[:,P_w]) with no handle and no allocation.
    Ti [W][n][n] = A^-T, idx int32 [W][k], rows [W][k][n], out [W] (all caller-owned CUDA
    tensors, contiguous; this wrapper creates no tensor either).  The call's scratch is a fixed
    1 MiB array in the library: W*k*k*itemsize beyond it raises LruxError (ELIMIT); calls that
    may overlap on the GPU race."""
    for t in (Ti, idx, rows, out):
        if not (t.is_cuda and t.is_contiguous()):
            raise ValueError("det_ratio_noalloc takes contiguous CUDA tensors")
    if idx.dtype != torch.int32 or rows.dtype != Ti.dtype or out.dtype != Ti.dtype:
        raise TypeError("idx must be int32; rows and out must have the dtype of Ti")
    W, n, k = int(Ti.shape[0]), int(Ti.shape[1]), int(idx.shape[1])
    if tuple(Ti.shape) != (W, n, n) or tuple(idx.shape) != (W, k) or tuple(rows.shape) != (W, k, n) \
            or out.numel() != W:
        raise ValueError("shape mismatch")
    _check(load_library().lrux_det_ratio_noalloc(W, n, k, _dt(Ti.dtype), _ptr(Ti), _ptr(idx), _ptr(rows),
                                                 _ptr(out), _stream(stream)))
    return out


def _optr(t):
    return None if t is None else _ptr(t)


def det_propose(seed, w0, step, Phi, occ, unocc, idx, upos, rows, d_step=None, stream=None):
    W, M, n = Phi.shape
    k = idx.shape[1]
    _check(load_library().lruxh_det_propose(seed, w0, step, W, n, M, k, _dt(Phi.dtype), _ptr(Phi),
                                            _ptr(occ), _ptr(unocc), _ptr(idx), _ptr(upos),
                                            _ptr(rows), _optr(d_step), _stream(stream)))


def pf_propose(seed, w0, step, F, occ, unocc, idx, upos, rows, d_step=None, stream=None):
    W, M, _ = F.shape
    n = occ.shape[1]
    k = idx.shape[1]
    _check(load_library().lruxh_pf_propose(seed, w0, step, W, n, M, k, _dt(F.dtype), _ptr(F),
                                           _ptr(occ), _ptr(unocc), _ptr(idx), _ptr(upos),
                                           _ptr(rows), _optr(d_step), _stream(stream)))


def decide(seed, w0, step, ratio, idx, upos, occ, unocc, mask, naccept, d_step=None, stream=None):
    """d_step: int64[2] device tensor ([0] step, [1] scratch = 0) read instead of ``step`` and
    advanced by one (CUDA-graph replay), or None."""
    W, n = occ.shape
    M = n + unocc.shape[1]
    k = idx.shape[1]
    _check(load_library().lruxh_decide(seed, w0, step, W, n, M, k, _dt(ratio.dtype), _ptr(ratio),
                                       _ptr(idx), _ptr(upos), _ptr(occ), _ptr(unocc), _ptr(mask),
                                       _ptr(naccept), _optr(d_step), _stream(stream)))
