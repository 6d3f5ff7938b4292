"""ctypes front end of the C oracle (oracle/lrux_oracle_c.c).

TEST INFRASTRUCTURE ONLY: same functions and return conventions as
``oracle/lrux_oracle.py`` (which stays as the by-eye checkable numpy statement and as a
cross-check), but compiled: plain C loops, float64 / complex128, no BLAS, OpenMP over
walkers in ``batch``.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
cpu_baseline / ``--impl reference`` legs may import this module.  It does not import
the product package and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build_oracle

_lib = None
_vp, _i32 = C.c_void_p, C.c_int32


class _Cfg(C.Structure):
    _fields_ = [(k, _i32) for k in ("kind", "n", "M", "k", "steps", "scratch_every", "delay", "final_scratch",
                                    "mark_step")]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build_oracle.build())
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def num_threads():
    return int(lib().orc_num_threads())


def _prep(A):
    A = np.asarray(A)
    cplx = np.iscomplexobj(A)
    return np.ascontiguousarray(A, dtype=np.complex128 if cplx else np.float64), ("z" if cplx else "d")


def _p(a):
    return a.ctypes.data_as(_vp) if a is not None else None


def _scalar(sfx):
    return np.zeros(1, np.complex128 if sfx == "z" else np.float64)


def _out(x, sfx):
    return complex(x) if sfx == "z" else float(x)


def slogdet(A):
    A, s = _prep(A)
    ph, la = _scalar(s), np.zeros(1)
    getattr(lib(), "orc_slogdet_" + s)(A.shape[0], _p(A), _p(ph), _p(la))
    return A.dtype.type(ph[0]), float(la[0])


def det(A):
    ph, la = slogdet(A)
    return ph * np.exp(la)


def inv(A):
    A, s = _prep(A)
    out = np.empty_like(A)
    if not getattr(lib(), "orc_inv_" + s)(A.shape[0], _p(A), _p(out)):
        raise np.linalg.LinAlgError("singular matrix in c_oracle.inv")
    return out


def slogpf(A):
    A, s = _prep(A)
    ph, la = _scalar(s), np.zeros(1)
    getattr(lib(), "orc_slogpf_" + s)(A.shape[0], _p(A), _p(ph), _p(la))
    return A.dtype.type(ph[0]), float(la[0])


def pf(A):
    ph, la = slogpf(A)
    return ph * np.exp(la)


def _common(*arrs):
    cplx = any(np.iscomplexobj(a) for a in arrs)
    dt = np.complex128 if cplx else np.float64
    return [np.ascontiguousarray(a, dtype=dt) for a in arrs], ("z" if cplx else "d")


def det_lru(Ainv, u, v, return_update=False):
    n = np.asarray(Ainv).shape[0]
    (Ainv, u, v), s = _common(Ainv, np.asarray(u).reshape(n, -1), np.asarray(v).reshape(n, -1))
    k = u.shape[1]
    r = _scalar(s)
    new = np.empty_like(Ainv) if return_update else None
    getattr(lib(), "orc_det_lru_" + s)(n, k, _p(Ainv), _p(u), _p(v), _p(r), _p(new))
    return (Ainv.dtype.type(r[0]), new) if return_update else Ainv.dtype.type(r[0])


def pf_lru(Ainv, u, return_update=False):
    n = np.asarray(Ainv).shape[0]
    (Ainv, u), s = _common(Ainv, np.asarray(u).reshape(n, -1))
    k = u.shape[1] // 2
    r = _scalar(s)
    new = np.empty_like(Ainv) if return_update else None
    getattr(lib(), "orc_pf_lru_" + s)(n, k, _p(Ainv), _p(u), _p(r), _p(new))
    return (Ainv.dtype.type(r[0]), new) if return_update else Ainv.dtype.type(r[0])


def pf_update_vectors(A_old_rows, A_new_rows, P, n):
    (o, nw), s = _common(np.asarray(A_old_rows), np.asarray(A_new_rows))
    k = len(P)
    Pa = np.ascontiguousarray(P, dtype=np.int32)
    u = np.empty((n, 2 * k), o.dtype)
    getattr(lib(), "orc_pf_update_vectors_" + s)(n, k, _p(o), _p(nw), _p(Pa), _p(u))
    return u


def batch(kind, orb, occ, unocc, P, J, xi, scratch_every=1, delay=0, final_scratch=True, threads=0,
          want_matrices=True, mark_step=None):
    """Trajectories of W independent walkers (OpenMP over walkers).

    orb [W][M][n] (det) or [W][M][M] (pf); occ [W][n], unocc [W][M-n] int32;
    P, J [steps][W][k] int32 and xi [steps][W] as ``workload.proposals`` returns them.
    Returns a list of W dicts with the keys of ``lrux_oracle.det_trajectory``.
    ``mark_step`` (timing only): each dict also carries ``seconds`` = the time that walker
    spent in steps >= mark_step (the O(n^3) initialisation and earlier steps left out).
    """
    orb, s = _prep(orb)
    occ = np.ascontiguousarray(occ, dtype=np.int32)
    unocc = np.ascontiguousarray(unocc, dtype=np.int32)
    W, n = occ.shape
    M = orb.shape[1]
    steps, _, k = np.asarray(P).shape
    Pw = np.ascontiguousarray(np.transpose(np.asarray(P, dtype=np.int32), (1, 0, 2)))
    Jw = np.ascontiguousarray(np.transpose(np.asarray(J, dtype=np.int32), (1, 0, 2)))
    xw = np.ascontiguousarray(np.asarray(xi, dtype=np.float64).T)
    dt = orb.dtype
    r_lemma = np.zeros((W, steps), dt)
    r_scratch = np.zeros((W, steps), dt)
    accepted = np.zeros((W, steps), np.uint8)
    near = np.zeros((W, steps), np.uint8)
    prob = np.zeros((W, steps))
    A = np.zeros((W, n, n), dt) if want_matrices else None
    Ainv = np.zeros((W, n, n), dt) if want_matrices else None
    occ_o, unocc_o = np.zeros_like(occ), np.zeros_like(unocc)
    amp, logs = np.zeros((W, 3), dt), np.zeros((W, 3))
    dur = np.zeros(W) if mark_step is not None else None
    cfg = _Cfg(0 if kind == "det" else 1, n, M, k, steps, int(scratch_every), int(delay), int(bool(final_scratch)),
               int(mark_step or 0))
    getattr(lib(), "orc_batch_" + s)(C.byref(cfg), W, int(threads), _p(orb), _p(occ), _p(unocc), _p(Pw), _p(Jw),
                                     _p(xw), _p(r_lemma), _p(r_scratch), _p(accepted), _p(near), _p(prob),
                                     _p(A), _p(Ainv), _p(occ_o), _p(unocc_o), _p(amp), _p(logs), _p(dur))
    out = []
    for w in range(W):
        out.append(dict(r_lemma=r_lemma[w], r_scratch=r_scratch[w], accepted=accepted[w].astype(bool),
                        near_tie=near[w].astype(bool), prob=prob[w],
                        A=A[w] if want_matrices else None, Ainv=Ainv[w] if want_matrices else None,
                        occ=occ_o[w], unocc=unocc_o[w],
                        phase=dt.type(amp[w, 0]), scratch_phase=dt.type(amp[w, 1]), init_phase=dt.type(amp[w, 2]),
                        logabs=float(logs[w, 0]), scratch_logabs=float(logs[w, 1]), init_logabs=float(logs[w, 2]),
                        seconds=float(dur[w]) if dur is not None else None))
    return out


def _one(kind, orb, occ, unocc, P, J, xi, scratch_every, delay):
    P = np.asarray(P)
    k = P.shape[1] if P.ndim == 2 else 1
    steps = len(xi)
    return batch(kind, np.asarray(orb)[None], np.asarray(occ)[None], np.asarray(unocc)[None],
                 P.reshape(steps, 1, k), np.asarray(J).reshape(steps, 1, k), np.asarray(xi).reshape(steps, 1),
                 scratch_every=scratch_every, delay=delay, final_scratch=True, threads=1)[0]


def det_trajectory(Phi, occ, unocc, P, J, xi, scratch_every=1, delay=0):
    """One walker; same contract as ``lrux_oracle.det_trajectory``."""
    return _one("det", Phi, occ, unocc, P, J, xi, scratch_every, delay)


def pf_trajectory(F, occ, unocc, P, J, xi, scratch_every=1, delay=0):
    """One walker; same contract as ``lrux_oracle.pf_trajectory``."""
    return _one("pf", F, occ, unocc, P, J, xi, scratch_every, delay)
