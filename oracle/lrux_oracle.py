"""CPU oracle for low-rank updates of determinants and Pfaffians.

TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct numpy (float64 /
complex128) restatement of what the hot path computes, written from
/root/reference/PAPER.md.  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s cpu_baseline / ``--impl reference`` legs may import this module.
It shares no code with the CUDA path (``paper_2602_05255_b200/csrc``) and does
not import the product package; inputs are passed in as arrays.

All ``.T`` below are plain transposes, never conjugate transposes, also for
complex data.

Parts:
  1. ``lu_factor`` / ``slogdet`` / ``inv``    partial-pivot LU (seed of A^-1, det A;
                                              PAPER.md:74-75, 97-98)
  2. ``slogpf`` / ``pf``                      Parlett-Reid with pivoting (PAPER.md:445
                                              leaves the algorithm open; reading 10)
  3. ``det_bruteforce`` / ``pf_bruteforce``   Leibniz sum; Eq. A.1
  4. ``det_lru`` / ``pf_lru``                 Eq. 2-5; Eq. 16-21
                                              
  5. ``DetCarrier`` / ``PfCarrier``           delayed updates Eq. 10-15
                                              and Eq. 25-28
  6. ``det_trajectory`` / ``pf_trajectory``   Metropolis chains of BASELINE.json configs

Pins: every function here is pinned in tests/test_oracle_pins.py against brute
force (n <= 8), the closed forms the paper prints (Eq. A.2, A.3, pf J), the
Pfaffian identities A.4-A.9, numpy.linalg as a library special case, the lemma
vs. from-scratch recomputation, A_t A_t^-1 = 1 and the telescoping product of
ratios.  No function is "parity unpinned".
"""
from __future__ import annotations

import itertools

import numpy as np

# ----------------------------------------------------------------------------
# 1. partial-pivot LU
# ----------------------------------------------------------------------------


def lu_factor(A):
    """Partial-pivot LU of a square matrix.

    Pivot = largest modulus in the column at or below the diagonal, lowest
    index on ties.  Returns (LU, perm, sign, ok):
    L (unit lower) and U packed in LU, ``perm`` the row order so that
    A[perm] = L U, ``sign`` = parity of the row swaps, ``ok`` False when a zero
    pivot was met (singular A).
    """
    LU = np.array(A, dtype=np.result_type(A, np.float64), copy=True)
    n = LU.shape[0]
    perm = np.arange(n)
    sign = 1.0
    ok = True
    for c in range(n):
        p = c + int(np.argmax(np.abs(LU[c:, c])))
        if LU[p, c] == 0:
            ok = False
            continue
        if p != c:
            LU[[c, p]] = LU[[p, c]]
            perm[[c, p]] = perm[[p, c]]
            sign = -sign
        LU[c + 1:, c] = LU[c + 1:, c] / LU[c, c]
        LU[c + 1:, c + 1:] = LU[c + 1:, c + 1:] - np.outer(LU[c + 1:, c], LU[c, c + 1:])
    return LU, perm, sign, ok


def slogdet(A):
    """(phase, log|det A|): phase = parity * prod U_ii/|U_ii|, logabs = sum log|U_ii|.
    Singular A gives (0, -inf)."""
    A = np.asarray(A)
    if A.shape[0] == 0:
        return A.dtype.type(1), 0.0
    LU, _, sign, ok = lu_factor(A)
    d = np.diag(LU)
    if not ok or np.any(d == 0):
        return LU.dtype.type(0), -np.inf
    phase = sign * np.prod(d / np.abs(d))
    return LU.dtype.type(phase), float(np.sum(np.log(np.abs(d))))


def det(A):
    ph, la = slogdet(A)
    return ph * np.exp(la)


def inv(A):
    """A^-1 by LU and n pairs of triangular solves (forward then backward)."""
    LU, perm, _, ok = lu_factor(A)
    n = LU.shape[0]
    if not ok or np.any(np.diag(LU) == 0):
        raise np.linalg.LinAlgError("singular matrix in oracle.inv")
    B = np.eye(n, dtype=LU.dtype)[perm]          # P * I
    Y = np.zeros_like(B)
    for i in range(n):                            # L Y = P I
        Y[i] = B[i] - LU[i, :i] @ Y[:i]
    X = np.zeros_like(B)
    for i in range(n - 1, -1, -1):                # U X = Y
        X[i] = (Y[i] - LU[i, i + 1:] @ X[i + 1:]) / LU[i, i]
    return X


# ----------------------------------------------------------------------------
# 2. Pfaffian by Parlett-Reid elimination with pivoting
# ----------------------------------------------------------------------------


def slogpf(A):
    """(phase, log|pf A|) of a skew-symmetric matrix, cf. lrux.slogpf.

    For j = 0,2,4,...: pivot p in [j+1,n) maximising |A[p][j]| (lowest index on
    ties); a simultaneous row+column swap j+1 <-> p flips the sign (Eq. A.5 with
    B a transposition); pf picks up the factor A[j][j+1] and the
    trailing block receives the Schur complement N + Q^T M^-1 Q of Eq. A.9
     with M = [[0,a],[-a,0]]:  A[j+2:,j+2:] += tau (x) c - c (x) tau,
    tau = A[j][j+2:]/a, c = A[j+2:][j+1].
    """
    A = np.array(A, dtype=np.result_type(A, np.float64), copy=True)
    n = A.shape[0]
    one = A.dtype.type(1)
    if n == 0:
        return one, 0.0
    if n % 2 == 1:
        return A.dtype.type(0), -np.inf
    phase = one
    logabs = 0.0
    for j in range(0, n - 1, 2):
        p = j + 1 + int(np.argmax(np.abs(A[j + 1:, j])))
        if p != j + 1:
            A[[j + 1, p], :] = A[[p, j + 1], :]
            A[:, [j + 1, p]] = A[:, [p, j + 1]]
            phase = -phase
        a = A[j, j + 1]
        if a == 0:
            return A.dtype.type(0), -np.inf
        phase = phase * (a / np.abs(a))
        logabs += float(np.log(np.abs(a)))
        if j + 2 < n:
            tau = A[j, j + 2:] / a
            c = A[j + 2:, j + 1].copy()
            A[j + 2:, j + 2:] = A[j + 2:, j + 2:] + np.outer(tau, c) - np.outer(c, tau)
    return A.dtype.type(phase), logabs


def pf(A):
    ph, la = slogpf(A)
    return ph * np.exp(la)


def skew_eye(k, dtype=np.float64):
    """J = [[0, 1],[-1, 0]] (2k x 2k), Eq. 17, lrux.skew_eye."""
    J = np.zeros((2 * k, 2 * k), dtype=dtype)
    J[:k, k:] = np.eye(k)
    J[k:, :k] = -np.eye(k)
    return J


def pf_skew_eye(k):
    """pf J = (-1)^(k(k-1)/2)."""
    return -1.0 if (k * (k - 1) // 2) % 2 else 1.0


# ----------------------------------------------------------------------------
# 3. brute force (n <= 8)
# ----------------------------------------------------------------------------


def _perm_sign(perm):
    inv_count = 0
    for i in range(len(perm)):
        for j in range(i + 1, len(perm)):
            inv_count += perm[i] > perm[j]
    return -1 if inv_count % 2 else 1


def det_bruteforce(A):
    """Leibniz sum over all n! permutations."""
    A = np.asarray(A)
    n = A.shape[0]
    total = 0
    for perm in itertools.permutations(range(n)):
        term = _perm_sign(perm)
        for i in range(n):
            term = term * A[i, perm[i]]
        total = total + term
    return total


def _pairings(items):
    if not items:
        yield []
        return
    i = items[0]
    for idx in range(1, len(items)):
        j = items[idx]
        rest = items[1:idx] + items[idx + 1:]
        for tail in _pairings(rest):
            yield [(i, j)] + tail


def pf_bruteforce(A):
    """Eq. A.1: sum over the (2n-1)!! partitions into pairs
    (i_k < j_k, i_1 < i_2 < ...) of sign(i_1 j_1 i_2 j_2 ...) prod A[i_k][j_k]."""
    A = np.asarray(A)
    n = A.shape[0]
    if n % 2:
        return 0
    total = 0
    for alpha in _pairings(list(range(n))):
        flat = [x for pair in alpha for x in pair]
        term = _perm_sign(flat)
        for (i, j) in alpha:
            term = term * A[i, j]
        total = total + term
    return total


# ----------------------------------------------------------------------------
# 4. low-rank updates: determinant (Eq. 2-5) and Pfaffian (Eq. 16-21)
# ----------------------------------------------------------------------------


def one_hot(idx, n, dtype=np.float64):
    """n x k matrix of one-hot columns e_{idx[a]} (Eq. 6, 8)."""
    idx = np.atleast_1d(idx)
    E = np.zeros((n, len(idx)), dtype=dtype)
    for a, p in enumerate(idx):
        E[p, a] = 1
    return E


def det_lru(Ainv, u, v, return_update=False):
    """lrux.det_lru.  A_t = A_{t-1} + v u^T.

    R = 1 + u^T A^-1 v (Eq. 4), r = det R (Eq. 3); with ``return_update``
    also A_t^-1 = A^-1 - A^-1 v R^-1 u^T A^-1 (Eq. 5).  u, v are n x k.
    """
    u = np.asarray(u).reshape(Ainv.shape[0], -1)
    v = np.asarray(v).reshape(Ainv.shape[0], -1)
    k = u.shape[1]
    R = np.eye(k, dtype=Ainv.dtype) + u.T @ Ainv @ v
    r = det(R)
    if not return_update:
        return r
    new = Ainv - (Ainv @ v) @ inv(R) @ (u.T @ Ainv)
    return r, new


def _skew_from_upper(G):
    up = np.triu(G, 1)
    return up - up.T


def pf_lru(Ainv, u, return_update=False):
    """lrux.pf_lru.  A_t = A_{t-1} - u J u^T, u is n x 2k.

    R = J + u^T A^-1 u (Eq. 20; Eq. 18 prints A without the inverse, a typo:
    DESIGN.md reading 1), r = pf R / pf J (Eq. 19).  R is built from its strict
    upper triangle and mirrored so that it is exactly skew (reading 8).  With
    ``return_update`` also A_t^-1 = A^-1 + (A^-1 u) R^-1 (A^-1 u)^T (Eq. 21) with an
    exactly skew R^-1 and an exactly skew result.
    """
    u = np.asarray(u).reshape(Ainv.shape[0], -1)
    k = u.shape[1] // 2
    R = skew_eye(k, Ainv.dtype) + _skew_from_upper(u.T @ Ainv @ u)
    r = pf(R) / pf_skew_eye(k)
    if not return_update:
        return r
    Rinv = inv(R)
    Rinv = (Rinv - Rinv.T) / 2
    a = Ainv @ u
    new = Ainv + _skew_from_upper(a @ Rinv @ a.T)
    return r, new


def pf_update_vectors(A_old_rows, A_new_rows, P, n):
    """u = (x, e) for replacing the rows AND columns P of a skew matrix
    (Eq. 23-24).

    ``A_old_rows[a]`` / ``A_new_rows[a]`` are row P[a] of A_{t-1} / A_t.  x[:,a] is
    the row delta; where replaced rows and columns cross, the delta is halved
    (reading 5) because -u J u^T = e x^T - x e^T counts that block twice;
    the diagonal entry multiplies A^-1[p][p] = 0 and is set to 0 (reading 6).
    """
    k = len(P)
    X = (np.asarray(A_new_rows) - np.asarray(A_old_rows)).T.copy()   # n x k
    for a in range(k):
        for b in range(k):
            X[P[b], a] = X[P[b], a] / 2
    return np.concatenate([X, one_hot(P, n, X.dtype)], axis=1)


# ----------------------------------------------------------------------------
# 5. delayed updates
# ----------------------------------------------------------------------------


class DetCarrier:
    """lrux.init_det_carrier / det_lru_delayed: A_0^-1 plus the
    delayed factors a_t (Eq. 10) and b_t (Eq. 11)."""

    def __init__(self, A, max_delay, Ainv=None):
        self.A0inv = inv(A) if Ainv is None else np.array(Ainv, copy=True)
        self.max_delay = int(max_delay)
        self.a = []
        self.b = []

    def lru(self, u, v, return_update=False):
        n = self.A0inv.shape[0]
        u = np.asarray(u).reshape(n, -1)
        v = np.asarray(v).reshape(n, -1)
        k = u.shape[1]
        R = np.eye(k, dtype=self.A0inv.dtype) + u.T @ self.A0inv @ v            # Eq. 13
        for a_t, b_t in zip(self.a, self.b):
            R = R - (u.T @ a_t) @ (b_t.T @ v)
        r = det(R)
        if not return_update:
            return r
        a = self.A0inv @ v                                                     # Eq. 14
        for a_t, b_t in zip(self.a, self.b):
            a = a - a_t @ (b_t.T @ v)
        b = self.A0inv.T @ u                                                   # Eq. 15
        for a_t, b_t in zip(self.a, self.b):
            b = b - b_t @ (a_t.T @ u)
        b = b @ inv(R).T
        self.a.append(a)
        self.b.append(b)
        if len(self.a) == self.max_delay:                                      # tau = T
            self.flush()
        return r

    def flush(self):
        for a_t, b_t in zip(self.a, self.b):                                   # Eq. 12
            self.A0inv = self.A0inv - a_t @ b_t.T
        self.a, self.b = [], []

    def inverse(self):
        out = self.A0inv.copy()
        for a_t, b_t in zip(self.a, self.b):
            out = out - a_t @ b_t.T
        return out


class PfCarrier:
    """lrux.init_pf_carrier / pf_lru_delayed: A_0^-1, a_t (Eq. 25)
    and R_t^-1."""

    def __init__(self, A, max_delay, Ainv=None):
        if Ainv is None:
            Ainv = inv(A)
            Ainv = (Ainv - Ainv.T) / 2
        self.A0inv = np.array(Ainv, copy=True)
        self.max_delay = int(max_delay)
        self.a = []
        self.Rinv = []

    def lru(self, u, return_update=False):
        n = self.A0inv.shape[0]
        u = np.asarray(u).reshape(n, -1)
        k = u.shape[1] // 2
        G = u.T @ self.A0inv @ u                                               # Eq. 27
        for a_t, Ri in zip(self.a, self.Rinv):
            ua = u.T @ a_t
            G = G + ua @ Ri @ ua.T
        R = skew_eye(k, self.A0inv.dtype) + _skew_from_upper(G)
        r = pf(R) / pf_skew_eye(k)
        if not return_update:
            return r
        a = self.A0inv @ u                                                     # Eq. 28 (u_tau)
        for a_t, Ri in zip(self.a, self.Rinv):
            a = a + a_t @ Ri @ (u.T @ a_t).T
        Rinv = inv(R)
        Rinv = (Rinv - Rinv.T) / 2
        self.a.append(a)
        self.Rinv.append(Rinv)
        if len(self.a) == self.max_delay:
            self.flush()
        return r

    def flush(self):
        for a_t, Ri in zip(self.a, self.Rinv):                                 # Eq. 26
            self.A0inv = self.A0inv + _skew_from_upper(a_t @ Ri @ a_t.T)
        self.a, self.Rinv = [], []

    def inverse(self):
        out = self.A0inv.copy()
        for a_t, Ri in zip(self.a, self.Rinv):
            out = out + _skew_from_upper(a_t @ Ri @ a_t.T)
        return out


# ----------------------------------------------------------------------------
# 6. Metropolis trajectories (BASELINE.json configs; SURVEY.md §8(c) part 4)
# ----------------------------------------------------------------------------

NEAR_TIE = 1e-8   # |xi - p| below this is logged as a near-tie (reading 15)


def metropolis_accept(r, xi):
    """accept iff xi < min(1, |r|^2), strictly; NaN ratio rejects (reading 12)."""
    a2 = float(np.real(r) ** 2 + np.imag(r) ** 2)
    if np.isnan(a2):
        return False, float("nan")
    p = min(1.0, a2)
    return bool(xi < p), p


def _quot(ph1, la1, ph0, la0):
    return (ph1 / ph0) * np.exp(la1 - la0)


def det_trajectory(Phi, occ, unocc, P, J, xi, scratch_every=1, delay=0, on_step=None):
    """One walker's chain of k-row replacements (BASELINE.json configs[0,1,3]).

    A = Phi[occ,:].  Step t proposes to put orbital unocc[J[t][a]] into slot
    P[t][a]: u = (new rows - old rows)^T, v = one-hot(P) (Eq. 8);
    ``r_lemma`` by Eq. 3-4, ``r_scratch`` = det A'/det A with both determinants
    recomputed by LU (every ``scratch_every`` steps, else NaN); accepted updates
    apply Eq. 5 naively (``delay`` = 0) or go through ``DetCarrier`` with
    max_delay = ``delay``.  The amplitude is tracked as (phase, log|det|).
    """
    Phi = np.asarray(Phi)
    occ = np.array(occ, copy=True)
    unocc = np.array(unocc, copy=True)
    n = len(occ)
    steps = len(xi)
    A = Phi[occ, :].copy()
    ph0, la0 = slogdet(A)
    phase, logabs = ph0, la0                 # tracked amplitude
    s_ph, s_la = ph0, la0                    # from-scratch amplitude of current A
    Ainv = inv(A)
    carrier = DetCarrier(A, delay, Ainv) if delay else None
    out = dict(r_lemma=np.zeros(steps, A.dtype), r_scratch=np.full(steps, np.nan, A.dtype),
               accepted=np.zeros(steps, bool), near_tie=np.zeros(steps, bool),
               prob=np.zeros(steps), init_phase=ph0, init_logabs=la0)
    for t in range(steps):
        p = [int(x) for x in P[t]]
        q = [int(unocc[j]) for j in J[t]]
        N = Phi[q, :]
        u = (N - A[p, :]).T
        v = one_hot(p, n, A.dtype)
        r = carrier.lru(u, v) if carrier else det_lru(Ainv, u, v)
        out["r_lemma"][t] = r
        A_new = A.copy()
        A_new[p, :] = N
        if scratch_every and (t % scratch_every == 0 or t == steps - 1):
            n_ph, n_la = slogdet(A_new)
            out["r_scratch"][t] = _quot(n_ph, n_la, s_ph, s_la)
        acc, prob = metropolis_accept(r, xi[t])
        out["accepted"][t] = acc
        out["prob"][t] = prob
        out["near_tie"][t] = abs(xi[t] - prob) < NEAR_TIE
        if acc:
            if carrier:
                carrier.lru(u, v, return_update=True)
            else:
                _, Ainv = det_lru(Ainv, u, v, return_update=True)
            A = A_new
            if scratch_every:                # from-scratch amplitude of the current A (checks only)
                s_ph, s_la = slogdet(A)
            phase = phase * (r / abs(r))
            logabs = logabs + float(np.log(abs(r)))
            for a in range(len(p)):
                occ[p[a]], unocc[J[t][a]] = unocc[J[t][a]], occ[p[a]]
        if on_step is not None:
            on_step(t)        # timing hook for bench.py; takes no part in the arithmetic
    if not scratch_every:
        s_ph, s_la = slogdet(A)              # amplitude of the final A, once
    out.update(A=A, Ainv=carrier.inverse() if carrier else Ainv, occ=occ, unocc=unocc,
               phase=phase, logabs=logabs, scratch_phase=s_ph, scratch_logabs=s_la)
    return out


def pf_trajectory(F, occ, unocc, P, J, xi, scratch_every=1, delay=0, on_step=None):
    """One walker's chain of k-orbital replacements in a Pfaffian state
    (BASELINE.json configs[2]).  A = F[occ][:,occ]; replacing the orbital in slot p
    changes row p and column p of A (Eq. 23-24); u from ``pf_update_vectors``;
    ratio by Eq. 19-20, update by Eq. 21 (or ``PfCarrier`` when ``delay`` > 0).
    """
    F = np.asarray(F)
    occ = np.array(occ, copy=True)
    unocc = np.array(unocc, copy=True)
    n = len(occ)
    steps = len(xi)
    A = F[np.ix_(occ, occ)].copy()
    ph0, la0 = slogpf(A)
    phase, logabs = ph0, la0
    s_ph, s_la = ph0, la0
    Ainv = inv(A)
    Ainv = (Ainv - Ainv.T) / 2
    carrier = PfCarrier(A, delay, Ainv) if delay else None
    out = dict(r_lemma=np.zeros(steps, A.dtype), r_scratch=np.full(steps, np.nan, A.dtype),
               accepted=np.zeros(steps, bool), near_tie=np.zeros(steps, bool),
               prob=np.zeros(steps), init_phase=ph0, init_logabs=la0)
    for t in range(steps):
        p = [int(x) for x in P[t]]
        occ_new = occ.copy()
        for a in range(len(p)):
            occ_new[p[a]] = unocc[J[t][a]]
        A_new = F[np.ix_(occ_new, occ_new)].copy()
        u = pf_update_vectors(A[p, :], A_new[p, :], p, n)
        r = carrier.lru(u) if carrier else pf_lru(Ainv, u)
        out["r_lemma"][t] = r
        if scratch_every and (t % scratch_every == 0 or t == steps - 1):
            n_ph, n_la = slogpf(A_new)
            out["r_scratch"][t] = _quot(n_ph, n_la, s_ph, s_la)
        acc, prob = metropolis_accept(r, xi[t])
        out["accepted"][t] = acc
        out["prob"][t] = prob
        out["near_tie"][t] = abs(xi[t] - prob) < NEAR_TIE
        if acc:
            if carrier:
                carrier.lru(u, return_update=True)
            else:
                _, Ainv = pf_lru(Ainv, u, return_update=True)
            A = A_new
            if scratch_every:                # from-scratch amplitude of the current A (checks only)
                s_ph, s_la = slogpf(A)
            phase = phase * (r / abs(r))
            logabs = logabs + float(np.log(abs(r)))
            for a in range(len(p)):
                occ[p[a]], unocc[J[t][a]] = unocc[J[t][a]], occ[p[a]]
        if on_step is not None:
            on_step(t)        # timing hook for bench.py; takes no part in the arithmetic
    if not scratch_every:
        s_ph, s_la = slogpf(A)               # amplitude of the final A, once
    out.update(A=A, Ainv=carrier.inverse() if carrier else Ainv, occ=occ, unocc=unocc,
               phase=phase, logabs=logabs, scratch_phase=s_ph, scratch_logabs=s_la)
    return out
