"""Pins for oracle/lrux_oracle.py against what the paper and the mathematics fix
(SURVEY.md §8(c) "What pins each part").  CPU only."""
import os

import numpy as np
import pytest

from oracle import c_oracle, lrux_oracle as pyorc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "pf_closed_forms.txt")


class _COracle:
    """The C oracle, with the helpers it does not restate (brute force, J, one-hot)
    taken from the numpy one: those are what BOTH implementations are pinned to."""

    def __getattr__(self, name):
        return getattr(c_oracle, name) if hasattr(c_oracle, name) else getattr(pyorc, name)


@pytest.fixture(params=["numpy", "c"])
def orc(request):
    return pyorc if request.param == "numpy" else _COracle()


def rand(rng, shape, cplx):
    x = rng.standard_normal(shape)
    if cplx:
        x = x + 1j * rng.standard_normal(shape)
    return x


def rand_skew(rng, n, cplx):
    g = rand(rng, (n, n), cplx)
    return np.triu(g, 1) - np.triu(g, 1).T


# ---------------------------------------------------------------- closed forms
def _golden_rows(tag):
    for line in open(GOLDEN):
        line = line.split("#")[0].split()
        if line and line[0] == tag:
            yield [float(x) for x in line[1:]]


def test_pf_closed_form_A2(orc):
    for a, exp in _golden_rows("A2"):
        assert orc.pf(np.array([[0, a], [-a, 0.0]])) == pytest.approx(exp, rel=1e-15)


def test_pf_closed_form_A3(orc):
    for a, b, c, d, e, f, exp in _golden_rows("A3"):
        A = np.array([[0, a, b, c], [-a, 0, d, e], [-b, -d, 0, f], [-c, -e, -f, 0.0]])
        assert orc.pf(A) == pytest.approx(exp, rel=1e-14, abs=1e-14)
        assert orc.pf_bruteforce(A) == pytest.approx(exp, rel=1e-14, abs=1e-14)


def test_pf_skew_eye(orc):
    for k, exp in _golden_rows("PFJ"):
        k = int(k)
        assert orc.pf_skew_eye(k) == exp
        assert orc.pf(orc.skew_eye(k)) == pytest.approx(exp, rel=1e-15)
        if 2 * k <= 8:
            assert orc.pf_bruteforce(orc.skew_eye(k)) == exp


# ---------------------------------------------------------------- brute force
@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7])
def test_lu_det_vs_leibniz(orc, n, cplx):
    rng = np.random.default_rng(100 + n)
    for _ in range(3):
        A = rand(rng, (n, n), cplx)
        assert orc.det(A) == pytest.approx(orc.det_bruteforce(A), rel=1e-12)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("n", [2, 4, 6, 8])
def test_parlett_reid_vs_matchings(orc, n, cplx):
    rng = np.random.default_rng(200 + n)
    for _ in range(3):
        A = rand_skew(rng, n, cplx)
        assert orc.pf(A) == pytest.approx(orc.pf_bruteforce(A), rel=1e-12)


def test_pf_pivoting_needed_case(orc):
    # A[0][1] = 0 forces a pivot swap; brute force fixes the sign
    A = np.array([[0, 0, 2, 1], [0, 0, 3, 5], [-2, -3, 0, 7], [-1, -5, -7, 0.0]])
    assert orc.pf(A) == pytest.approx(orc.pf_bruteforce(A), rel=1e-14)
    assert orc.pf(A) == pytest.approx(0 * 7 - 2 * 5 + 1 * 3)


def test_pf_odd_and_singular(orc):
    assert orc.pf(np.zeros((3, 3))) == 0
    assert orc.pf(np.zeros((4, 4))) == 0
    assert orc.det(np.zeros((3, 3))) == 0
    assert orc.det(np.ones((3, 3))) == pytest.approx(0, abs=1e-15)


# ---------------------------------------------------------------- library / textbook
@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("n", [3, 17, 64])
def test_lu_vs_numpy_linalg(orc, n, cplx):
    rng = np.random.default_rng(300 + n)
    A = rand(rng, (n, n), cplx)
    ph, la = orc.slogdet(A)
    s, l = np.linalg.slogdet(A)
    assert ph == pytest.approx(s, rel=1e-11)
    assert la == pytest.approx(l, rel=1e-12)
    assert np.allclose(orc.inv(A), np.linalg.inv(A), rtol=1e-9, atol=1e-11)
    assert np.allclose(orc.inv(A) @ A, np.eye(n), atol=1e-10)


def test_det_triangular_and_product(orc):
    rng = np.random.default_rng(5)
    U = np.triu(rng.standard_normal((6, 6)))
    assert orc.det(U) == pytest.approx(np.prod(np.diag(U)), rel=1e-13)
    A, B = rng.standard_normal((2, 7, 7))
    assert orc.det(A @ B) == pytest.approx(orc.det(A) * orc.det(B), rel=1e-11)
    # a row swap flips the sign
    A2 = A.copy()
    A2[[0, 3]] = A2[[3, 0]]
    assert orc.det(A2) == pytest.approx(-orc.det(A), rel=1e-12)


# ---------------------------------------------------------------- Pfaffian identities A.4-A.9
@pytest.mark.parametrize("cplx", [False, True])
def test_pf_identities(orc, cplx):
    rng = np.random.default_rng(7)
    n = 10
    A = rand_skew(rng, n, cplx)
    B = rand(rng, (n, n), cplx)
    assert orc.pf(A) ** 2 == pytest.approx(orc.det(A), rel=1e-10)                       # A.4
    assert orc.pf(B @ A @ B.T) == pytest.approx(orc.det(B) * orc.pf(A), rel=1e-9)       # A.5
    m = 5
    G = rand(rng, (m, m), cplx)
    Z = np.zeros((m, m))
    blk = np.block([[Z, G], [-G.T, Z]])
    assert orc.pf(blk) == pytest.approx((-1) ** (m * (m - 1) // 2) * orc.det(G), rel=1e-10)   # A.6
    A2 = rand_skew(rng, 6, cplx)
    Zr = np.zeros((n, 6))
    assert orc.pf(np.block([[A, Zr], [Zr.T, A2]])) == pytest.approx(orc.pf(A) * orc.pf(A2), rel=1e-10)  # A.7
    # A.8 with C skew invertible (2k x 2k), B n x 2k
    k2 = 4
    C = rand_skew(rng, k2, cplx)
    Bm = rand(rng, (n, k2), cplx)
    Cinv = np.linalg.inv(C)
    lhs = orc.pf(A + Bm @ C @ Bm.T) / orc.pf(A)
    Ai = np.linalg.inv(A)
    S = Cinv + Bm.T @ Ai @ Bm
    S = (S - S.T) / 2
    Ci = (Cinv - Cinv.T) / 2
    assert lhs == pytest.approx(orc.pf(S) / orc.pf(Ci), rel=1e-9)
    # A.9
    Mb, Nb = rand_skew(rng, 4, cplx), rand_skew(rng, 6, cplx)
    Q = rand(rng, (4, 6), cplx)
    full = np.block([[Mb, Q], [-Q.T, Nb]])
    S1 = Nb + Q.T @ np.linalg.inv(Mb) @ Q
    S2 = Mb + Q @ np.linalg.inv(Nb) @ Q.T
    assert orc.pf(full) == pytest.approx(orc.pf(Mb) * orc.pf((S1 - S1.T) / 2), rel=1e-9)
    assert orc.pf(full) == pytest.approx(orc.pf(Nb) * orc.pf((S2 - S2.T) / 2), rel=1e-9)


# ---------------------------------------------------------------- lemma / Woodbury
@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("k", [1, 2, 3])
def test_det_lemma_dense(orc, k, cplx):
    """PAPER.md:69-85 recipe: det A * r == det(A + v u^T); Eq. 5 gives the inverse."""
    rng = np.random.default_rng(10 + k)
    n = 6
    A = rand(rng, (n, n), cplx)
    u, v = rand(rng, (n, k), cplx), rand(rng, (n, k), cplx)
    Ainv = np.linalg.inv(A)
    r, new = orc.det_lru(Ainv, u, v, return_update=True)
    assert r == pytest.approx(orc.det_bruteforce(A + v @ u.T) / orc.det_bruteforce(A), rel=1e-10)
    assert np.allclose(new @ (A + v @ u.T), np.eye(n), atol=1e-9)
    if k == 1:   # textbook Sherman-Morrison
        assert r == pytest.approx(1 + (u.T @ Ainv @ v)[0, 0], rel=1e-13)
        sm = Ainv - (Ainv @ v @ u.T @ Ainv) / (1 + u.T @ Ainv @ v)
        assert np.allclose(new, sm, rtol=1e-11, atol=1e-13)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("k", [1, 2])
def test_pf_lemma_dense(orc, k, cplx):
    """PAPER.md:250-267 recipe: pf A * r == pf(A - u J u^T); Eq. 21 gives the inverse."""
    rng = np.random.default_rng(20 + k)
    n = 8
    A = rand_skew(rng, n, cplx)
    u = rand(rng, (n, 2 * k), cplx)
    Ainv = np.linalg.inv(A)
    Ainv = (Ainv - Ainv.T) / 2
    A1 = A - u @ orc.skew_eye(k) @ u.T
    r, new = orc.pf_lru(Ainv, u, return_update=True)
    assert r == pytest.approx(orc.pf_bruteforce(A1) / orc.pf_bruteforce(A), rel=1e-10)
    assert np.allclose(new @ A1, np.eye(n), atol=1e-9)
    assert np.array_equal(new, -new.T)
    if k == 1:   # Eq. 22
        x, y = u[:, :1], u[:, 1:]
        ax, ay = Ainv @ x, Ainv @ y
        e22 = Ainv + (ay @ ax.T - ax @ ay.T) / r
        assert np.allclose(new, e22, rtol=1e-11, atol=1e-13)
        # with y = e_p and x_p = 0: r = 1 + x^T A^-1 e_p
        xe = rand(rng, (n,), cplx)
        xe[3] = 0
        ue = np.stack([xe, np.eye(n)[3]], axis=1)
        assert orc.pf_lru(Ainv, ue) == pytest.approx(1 + xe @ Ainv[:, 3], rel=1e-12)


@pytest.mark.parametrize("k", [1, 2, 3])
def test_pf_update_vectors_reproduce_row_col_replacement(orc, k):
    """Reading 5: A - u J u^T must equal A with rows and columns P replaced."""
    rng = np.random.default_rng(30 + k)
    n = 8
    A = rand_skew(rng, n, False)
    A1 = A.copy()
    P = list(rng.choice(n, k, replace=False))
    newrows = rand(rng, (k, n), False)
    for a, p in enumerate(P):
        A1[p, :] = newrows[a]
        A1[:, p] = -newrows[a]
    for a, p in enumerate(P):     # make the crossing block consistent and skew
        for b, q in enumerate(P):
            if a < b:
                A1[q, p] = -A1[p, q]
            if a == b:
                A1[p, p] = 0
    u = orc.pf_update_vectors(A[P, :], A1[P, :], P, n)
    assert np.allclose(A - u @ orc.skew_eye(k) @ u.T, A1, atol=1e-14)
    Ainv = np.linalg.inv(A)
    Ainv = (Ainv - Ainv.T) / 2
    assert orc.pf_lru(Ainv, u) == pytest.approx(orc.pf_bruteforce(A1) / orc.pf_bruteforce(A), rel=1e-10)


# ---------------------------------------------------------------- C oracle == numpy oracle
@pytest.mark.parametrize("cplx", [False, True])
def test_c_oracle_agrees_with_numpy_oracle(cplx):
    """Two independent restatements of the same definitions (different language, different
    summation order) agree to rounding on every shared function."""
    rng = np.random.default_rng(77)
    for n in (1, 2, 5, 12, 40):
        A = rand(rng, (n, n), cplx)
        (p1, l1), (p2, l2) = pyorc.slogdet(A), c_oracle.slogdet(A)
        assert p1 == pytest.approx(p2, abs=1e-11) and l1 == pytest.approx(l2, abs=1e-11)
        assert np.allclose(pyorc.inv(A), c_oracle.inv(A), rtol=1e-9, atol=1e-11)
        k = min(3, n)
        u, v = rand(rng, (n, k), cplx), rand(rng, (n, k), cplx)
        Ai = np.linalg.inv(A)
        r1, n1 = pyorc.det_lru(Ai, u, v, True)
        r2, n2 = c_oracle.det_lru(Ai, u, v, True)
        assert r1 == pytest.approx(r2, rel=1e-11)
        assert np.allclose(n1, n2, rtol=1e-9, atol=1e-11)
    for n in (2, 6, 12, 40):
        A = rand_skew(rng, n, cplx)
        (p1, l1), (p2, l2) = pyorc.slogpf(A), c_oracle.slogpf(A)
        assert p1 == pytest.approx(p2, abs=1e-11) and l1 == pytest.approx(l2, abs=1e-11)
        k = min(2, n // 2)
        u = rand(rng, (n, 2 * k), cplx)
        Ai = np.linalg.inv(A)
        Ai = (Ai - Ai.T) / 2
        r1, n1 = pyorc.pf_lru(Ai, u, True)
        r2, n2 = c_oracle.pf_lru(Ai, u, True)
        assert r1 == pytest.approx(r2, rel=1e-10)
        assert np.allclose(n1, n2, rtol=1e-8, atol=1e-10)
        assert np.array_equal(n2, -n2.T)
    assert c_oracle.slogdet(np.zeros((3, 3)))[1] == -np.inf
    assert c_oracle.slogpf(np.zeros((4, 4)))[1] == -np.inf
    with pytest.raises(np.linalg.LinAlgError):
        c_oracle.inv(np.zeros((3, 3)))
