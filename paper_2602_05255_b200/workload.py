"""Seeded synthetic workload generator (shared by tests, bench, oracle callers).

This module holds NONE of the method's arithmetic (no determinant, Pfaffian,
lemma or Woodbury step): it only turns (seed, walker, stream, counter) into
reproducible random inputs shaped like the paper's workloads, which are random
matrices batched over walkers.  The recipe
is the one SURVEY.md §8(d) fixes and DESIGN.md §4 restates.

Counter-based generator
-----------------------
``rnd64(seed, w, stream, ctr)`` is a pure function built from the splitmix64
finaliser.  The CUDA harness (csrc/lrux_harness.cu) re-implements exactly the
same integer function for the per-step proposal draws, so both sides consume
identical integers; everything floating point derived from it on the host
(Gaussians by Box-Muller) is uploaded as bytes.

* uniform in [0,1)   = top 53 bits * 2**-53
* integer in [0,m)   = high word of the 64x64 product with m  (m < 2**32)
* standard normal    = sqrt(-2 ln u1) cos(2 pi u2), u1 = (top53(ctr 2c)+1)*2**-53,
                       u2 = top53(ctr 2c+1)*2**-53   (one normal per counter c)

Streams: 0 matrix entries, 1 initial occupation, 2 slot draws, 3 orbital draws,
4 acceptance uniform.
"""
from __future__ import annotations

import numpy as np

BASE_SEED = 260205255  # seed_c = BASE_SEED + c for BASELINE.json config c in 1..5

STREAM_MATRIX = 0
STREAM_OCC = 1
STREAM_SLOT = 2
STREAM_ORB = 3
STREAM_ACCEPT = 4

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_C_STREAM = np.uint64(0xD1342543DE82EF95)
_MASK32 = np.uint64(0xFFFFFFFF)


def _u64(x):
    return np.asarray(x).astype(np.uint64)


def mix64(z):
    """splitmix64 finaliser on uint64 arrays (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        z = _u64(z)
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def rnd64(seed, w, stream, ctr):
    """64 random bits as a pure function of (seed, walker, stream, counter)."""
    with np.errstate(over="ignore"):
        h = mix64(_u64(seed) ^ (_u64(stream) * _C_STREAM))
        h = mix64(h + _u64(w) * _GOLDEN)
        return mix64(h + (_u64(ctr) + np.uint64(1)) * _GOLDEN)


def to_uniform(bits):
    """[0,1) double from the top 53 bits."""
    return (_u64(bits) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def to_below(bits, m):
    """Integer in [0,m): high 64 bits of bits*m, for m < 2**32."""
    bits = _u64(bits)
    m = _u64(m)
    hi = bits >> np.uint64(32)
    lo = bits & _MASK32
    with np.errstate(over="ignore"):
        return ((hi * m + ((lo * m) >> np.uint64(32))) >> np.uint64(32)).astype(np.int64)


def normal(seed, w, stream, ctr):
    """Standard normals (Box-Muller, host libm), one per counter value."""
    ctr = _u64(ctr)
    b1 = rnd64(seed, w, stream, ctr * np.uint64(2))
    b2 = rnd64(seed, w, stream, ctr * np.uint64(2) + np.uint64(1))
    u1 = ((b1 >> np.uint64(11)).astype(np.float64) + 1.0) * (2.0 ** -53)
    u2 = to_uniform(b2)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


# ----------------------------------------------------------------------------
# matrices
# ----------------------------------------------------------------------------
def orbital_matrix(seed, w, M, n, var, complex_=False):
    """Phi (M x n) for walker w: iid N(0,var) entries, counter = row-major index.

    Complex: real part from counters [0, M*n), imaginary part from
    [M*n, 2*M*n), each N(0,var) (BASELINE.json configs[3]).
    """
    cnt = np.arange(M * n, dtype=np.uint64)
    re = normal(seed, w, STREAM_MATRIX, cnt).reshape(M, n) * np.sqrt(var)
    if not complex_:
        return re
    im = normal(seed, w, STREAM_MATRIX, cnt + np.uint64(M * n)).reshape(M, n) * np.sqrt(var)
    return re + 1j * im


def pairing_matrix(seed, w, M, var, complex_=False):
    """Skew-symmetric F (M x M): F[i][j], i<j iid N(0,var) with counter i*M+j;
    F[j][i] = -F[i][j]; zero diagonal (BASELINE.json configs[2])."""
    cnt = np.arange(M * M, dtype=np.uint64)
    g = normal(seed, w, STREAM_MATRIX, cnt).reshape(M, M) * np.sqrt(var)
    if complex_:
        g = g + 1j * normal(seed, w, STREAM_MATRIX, cnt + np.uint64(M * M)).reshape(M, M) * np.sqrt(var)
    up = np.triu(g, 1)
    return up - up.T


def initial_occupation(seed, w, M, n):
    """Fisher-Yates shuffle of [0,M) driven by stream 1; occ = first n entries in
    shuffled order (never re-sorted), unocc = the rest."""
    perm = np.arange(M, dtype=np.int32)
    for i in range(M - 1, 0, -1):
        j = int(to_below(rnd64(seed, w, STREAM_OCC, M - 1 - i), i + 1))
        perm[i], perm[j] = perm[j], perm[i]
    return perm[:n].copy(), perm[n:].copy()


# ----------------------------------------------------------------------------
# per-step proposal draws
# ----------------------------------------------------------------------------
def _distinct(seed, ws, stream, step, k, m):
    """k distinct values in [0,m) per walker: draw rho_a in [0, m-a) with
    counter step*k+a and skip over previously chosen values in ascending
    order.  ``ws`` is an array of walker ids; returns int64 [len(ws)][k]."""
    ws = np.atleast_1d(np.asarray(ws, dtype=np.uint64))
    out = np.zeros((len(ws), k), np.int64)
    for a in range(k):
        rho = to_below(rnd64(seed, ws, stream, np.uint64(step * k + a)), m - a)
        if a:
            prev = np.sort(out[:, :a], axis=1)
            for c in range(a):
                rho = rho + (rho >= prev[:, c])
        out[:, a] = rho
    return out


def proposal(seed, w, step, n, M, k):
    """(slots P[k], positions J[k] in unocc, acceptance uniform xi) for one
    walker and step.  Pairing is in draw order: slot P[a] receives orbital
    unocc[J[a]]; on accept the caller swaps occ[P[a]] <-> unocc[J[a]]."""
    P = _distinct(seed, [w], STREAM_SLOT, step, k, n)[0]
    J = _distinct(seed, [w], STREAM_ORB, step, k, M - n)[0]
    xi = float(to_uniform(rnd64(seed, w, STREAM_ACCEPT, step)))
    return [int(x) for x in P], [int(x) for x in J], xi


def proposals(seed, W, steps, n, M, k, walkers=None):
    """Arrays P[steps][W'][k], J[steps][W'][k] (int32) and xi[steps][W'] for the
    listed walkers (default all W)."""
    ws = np.arange(W, dtype=np.uint64) if walkers is None else np.asarray(list(walkers), dtype=np.uint64)
    P = np.zeros((steps, len(ws), k), np.int32)
    J = np.zeros((steps, len(ws), k), np.int32)
    xi = np.zeros((steps, len(ws)), np.float64)
    for t in range(steps):
        P[t] = _distinct(seed, ws, STREAM_SLOT, t, k, n)
        J[t] = _distinct(seed, ws, STREAM_ORB, t, k, M - n)
        xi[t] = to_uniform(rnd64(seed, ws, STREAM_ACCEPT, np.uint64(t)))
    return P, J, xi


# ----------------------------------------------------------------------------
# device-side generation for full-size bench inputs (torch ops only: plumbing)
# ----------------------------------------------------------------------------
def _t_mix64(z):
    import torch  # local: the module must import without torch

    m1 = -4658895280553007687  # 0xBF58476D1CE4E5B9 as int64
    m2 = -7723592293110705685  # 0x94D049BB133111EB as int64
    z = (z ^ ((z >> 30) & ((1 << 34) - 1))) * m1
    z = (z ^ ((z >> 27) & ((1 << 37) - 1))) * m2
    return z ^ ((z >> 31) & ((1 << 33) - 1))


def _t_rnd64(seed, w, stream, ctr):
    import torch

    golden = -7046029254386353131  # 0x9E3779B97F4A7C15
    cs = -3372029247567499371  # 0xD1342543DE82EF95
    h = _t_mix64(torch.as_tensor(np.int64(np.uint64(seed).astype(np.int64)), device=ctr.device)
                 ^ (torch.as_tensor(stream, dtype=torch.int64, device=ctr.device) * cs))
    h = _t_mix64(h + w * golden)
    return _t_mix64(h + (ctr + 1) * golden)


def _t_top53(bits):
    return ((bits >> 11) & ((1 << 53) - 1)).to(dtype=__import__("torch").float64)


def normal_torch(seed, w, stream, ctr):
    """Same integers as ``normal``; log/cos/sqrt by torch on ``ctr.device`` (may
    differ from host libm in the last ulp: full-size parity replays downloaded
    bytes)."""
    import torch

    b1 = _t_rnd64(seed, w, stream, ctr * 2)
    b2 = _t_rnd64(seed, w, stream, ctr * 2 + 1)
    u1 = (_t_top53(b1) + 1.0) * (2.0 ** -53)
    u2 = _t_top53(b2) * (2.0 ** -53)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * np.pi * u2)


def orbital_matrices_torch(seed, w0, W, M, n, var, device, complex_=False, chunk=64):
    """Phi[W][M][n] for walkers w0..w0+W on ``device`` (float64 or complex128)."""
    import torch

    out = torch.empty((W, M, n), dtype=torch.complex128 if complex_ else torch.float64, device=device)
    cnt = torch.arange(M * n, dtype=torch.int64, device=device)
    s = float(np.sqrt(var))
    chunk = max(1, min(chunk, (1 << 27) // (M * n)))      # bound the temporaries
    for c0 in range(0, W, chunk):
        c1 = min(W, c0 + chunk)
        w = torch.arange(w0 + c0, w0 + c1, dtype=torch.int64, device=device)[:, None]
        re = normal_torch(seed, w, STREAM_MATRIX, cnt[None, :]).reshape(c1 - c0, M, n) * s
        if complex_:
            im = normal_torch(seed, w, STREAM_MATRIX, cnt[None, :] + M * n).reshape(c1 - c0, M, n) * s
            out[c0:c1] = torch.complex(re, im)
        else:
            out[c0:c1] = re
    return out


def pairing_matrices_torch(seed, w0, W, M, var, device, chunk=64):
    """F[W][M][M] skew-symmetric (float64) for walkers w0..w0+W on ``device``."""
    import torch

    out = torch.empty((W, M, M), dtype=torch.float64, device=device)
    cnt = torch.arange(M * M, dtype=torch.int64, device=device)
    s = float(np.sqrt(var))
    chunk = max(1, min(chunk, (1 << 27) // (M * M)))      # bound the temporaries (~10 arrays of chunk*M*M*8 B)
    for c0 in range(0, W, chunk):
        c1 = min(W, c0 + chunk)
        w = torch.arange(w0 + c0, w0 + c1, dtype=torch.int64, device=device)[:, None]
        g = normal_torch(seed, w, STREAM_MATRIX, cnt[None, :]).reshape(c1 - c0, M, M) * s
        up = torch.triu(g, 1)
        out[c0:c1] = up - up.transpose(1, 2)
    return out


def initial_occupations(seed, W, M, n, w0=0):
    """Vectorised over walkers; identical to ``initial_occupation`` per walker."""
    ws = np.arange(w0, w0 + W, dtype=np.uint64)
    perm = np.tile(np.arange(M, dtype=np.int32), (W, 1))
    rows = np.arange(W)
    for i in range(M - 1, 0, -1):
        j = to_below(rnd64(seed, ws, STREAM_OCC, np.uint64(M - 1 - i)), i + 1)
        pi = perm[rows, i].copy()
        perm[rows, i] = perm[rows, j]
        perm[rows, j] = pi
    return perm[:, :n].copy(), perm[:, n:].copy()
