"""Pins for the oracle's delayed carriers and Metropolis trajectory drivers:
the paper's own recipes (tracked amplitude vs. recomputed, PAPER.md:199-219,
371-392), delayed == immediate (Eq. 12 / Eq. 26), the telescoping product of
ratios (Eq. 3) and A_t A_t^-1 = 1.  CPU only."""
import numpy as np
import pytest

from oracle import c_oracle, lrux_oracle as pyorc
from paper_2602_05255_b200 import workload as wl

orc = pyorc     # the carrier objects exist in the numpy oracle only; the C carriers are pinned
                # through the delayed trajectories below and by C == numpy


@pytest.fixture(params=["numpy", "c"])
def traj(request):
    return pyorc if request.param == "numpy" else c_oracle


def rand(rng, shape, cplx):
    x = rng.standard_normal(shape)
    if cplx:
        x = x + 1j * rng.standard_normal(shape)
    return x


@pytest.mark.parametrize("cplx", [False, True])
def test_det_delayed_recipe(cplx):
    """n=10, max_delay=4, 20 one-hot row updates; tracked det
    equals the recomputed det after every step, and equals the immediate path."""
    rng = np.random.default_rng(42)
    n, T = 10, 4
    A = rand(rng, (n, n), cplx)
    car = orc.DetCarrier(A, T)
    Ainv = orc.inv(A)
    detA = orc.det(A)
    for i in range(20):
        u = rand(rng, (n,), cplx)
        p = int(rng.integers(n))
        v = orc.one_hot([p], n, A.dtype)
        r_imm, Ainv = orc.det_lru(Ainv, u[:, None], v, return_update=True)
        assert car.lru(u[:, None], v) == pytest.approx(r_imm, rel=1e-9)
        r = car.lru(u[:, None], v, return_update=True)
        assert len(car.a) == (i + 1) % T
        detA = detA * r
        A[p] += u
        assert detA == pytest.approx(orc.det(A), rel=1e-8)
        assert np.allclose(car.inverse(), Ainv, rtol=1e-7, atol=1e-9)
    assert np.allclose(car.inverse() @ A, np.eye(n), atol=1e-8)


@pytest.mark.parametrize("cplx", [False, True])
@pytest.mark.parametrize("k", [1, 2])
def test_pf_delayed_recipe(k, cplx):
    """n=10, max_delay=4, 20 row+column updates."""
    rng = np.random.default_rng(43 + k)
    n, T = 10, 4
    g = rand(rng, (n, n), cplx)
    A = (g - g.T) / 2
    car = orc.PfCarrier(A, T)
    Ainv = car.A0inv.copy()
    pfA = orc.pf(A)
    for i in range(20):
        P = list(rng.choice(n, k, replace=False))
        A1 = A.copy()
        for p in P:
            x = rand(rng, (n,), cplx)
            x[p] = 0
            A1[p, :] += x
            A1[:, p] -= x
        u = orc.pf_update_vectors(A[P, :], A1[P, :], P, n)
        assert np.allclose(A - u @ orc.skew_eye(k) @ u.T, A1, atol=1e-13)
        r_imm, Ainv = orc.pf_lru(Ainv, u, return_update=True)
        r = car.lru(u, return_update=True)
        assert r == pytest.approx(r_imm, rel=1e-8)
        pfA = pfA * r
        A = A1
        assert pfA == pytest.approx(orc.pf(A), rel=1e-7)
        assert np.allclose(car.inverse(), Ainv, rtol=1e-6, atol=1e-8)
    assert np.allclose(car.inverse() @ A, np.eye(n), atol=1e-7)


def _config1():
    seed = wl.BASE_SEED + 1
    n, M, k, steps = 32, 64, 1, 200
    Phi = wl.orbital_matrix(seed, 0, M, n, 1.0 / n)
    occ, unocc = wl.initial_occupation(seed, 0, M, n)
    P, J, xi = wl.proposals(seed, 1, steps, n, M, k)
    return Phi, occ, unocc, P[:, 0], J[:, 0], xi[:, 0]


def test_det_trajectory_config1(traj):
    """BASELINE.json configs[0]: 200 steps, k=1, n=32."""
    Phi, occ, unocc, P, J, xi = _config1()
    tr = traj.det_trajectory(Phi, occ, unocc, P, J, xi, scratch_every=1)
    acc = tr["accepted"]
    assert 0.2 < acc.mean() < 0.6          # SURVEY probe: ~0.36
    # lemma == from-scratch ratio at every step (Eq. 2)
    np.testing.assert_allclose(tr["r_lemma"], tr["r_scratch"], rtol=1e-8)
    # telescoping product (Eq. 3): tracked amplitude == det A_T recomputed
    assert tr["phase"] == tr["scratch_phase"]
    assert tr["logabs"] == pytest.approx(tr["scratch_logabs"], abs=1e-9)
    assert np.array_equal(tr["A"], Phi[tr["occ"], :])
    assert np.allclose(tr["A"] @ tr["Ainv"], np.eye(32), atol=1e-9)
    assert sorted(list(tr["occ"]) + list(tr["unocc"])) == list(range(64))
    # delayed path takes the same decisions and ends in the same inverse
    td = traj.det_trajectory(Phi, occ, unocc, P, J, xi, scratch_every=0, delay=4)
    assert np.array_equal(td["accepted"], acc)
    np.testing.assert_allclose(td["r_lemma"], tr["r_lemma"], rtol=1e-8)
    assert np.allclose(td["Ainv"], tr["Ainv"], rtol=1e-7, atol=1e-9)


@pytest.mark.parametrize("k", [2, 4])
def test_det_trajectory_complex_k(traj, k):
    seed = wl.BASE_SEED + 4
    n, M, steps = 16, 32, 60
    Phi = wl.orbital_matrix(seed, 3, M, n, 1.0 / (2 * n), complex_=True)
    occ, unocc = wl.initial_occupation(seed, 3, M, n)
    P, J, xi = wl.proposals(seed, 4, steps, n, M, k, walkers=[3])
    tr = traj.det_trajectory(Phi, occ, unocc, P[:, 0], J[:, 0], xi[:, 0])
    assert tr["accepted"].sum() > 3
    np.testing.assert_allclose(tr["r_lemma"], tr["r_scratch"], rtol=1e-7)
    assert tr["phase"] == pytest.approx(tr["scratch_phase"], abs=1e-9)
    assert tr["logabs"] == pytest.approx(tr["scratch_logabs"], abs=1e-9)
    assert np.allclose(tr["A"] @ tr["Ainv"], np.eye(n), atol=1e-8)


@pytest.mark.parametrize("k,delay", [(1, 0), (2, 0), (1, 3), (2, 3)])
def test_pf_trajectory(traj, k, delay):
    """BASELINE.json configs[2] shape at n=16: F skew 32x32, k orbital swaps."""
    seed = wl.BASE_SEED + 3
    n, M, steps = 16, 32, 80
    F = wl.pairing_matrix(seed, 1, M, 1.0 / n)
    assert np.array_equal(F, -F.T)
    occ, unocc = wl.initial_occupation(seed, 1, M, n)
    P, J, xi = wl.proposals(seed, 2, steps, n, M, k, walkers=[1])
    tr = traj.pf_trajectory(F, occ, unocc, P[:, 0], J[:, 0], xi[:, 0], delay=delay)
    assert tr["accepted"].sum() > 5
    np.testing.assert_allclose(tr["r_lemma"], tr["r_scratch"], rtol=1e-7)
    assert tr["phase"] == tr["scratch_phase"]
    assert tr["logabs"] == pytest.approx(tr["scratch_logabs"], abs=1e-8)
    assert np.array_equal(tr["A"], F[np.ix_(tr["occ"], tr["occ"])])
    assert np.allclose(tr["A"] @ tr["Ainv"], np.eye(n), atol=1e-8)
    assert np.array_equal(tr["Ainv"], -tr["Ainv"].T)


def test_metropolis_rule():
    assert orc.metropolis_accept(2.0, 0.999)[0]
    assert orc.metropolis_accept(0.5, 0.2499)[0]
    assert not orc.metropolis_accept(0.5, 0.25)[0]          # strict
    assert not orc.metropolis_accept(float("nan"), 0.0)[0]  # NaN rejects
    assert orc.metropolis_accept(0.3 + 0.4j, 0.2499)[0]
    assert not orc.metropolis_accept(0.3 + 0.4j, 0.2501)[0]


@pytest.mark.parametrize("kind,k,delay,cplx", [("det", 2, 0, False), ("det", 3, 5, True), ("det", 1, 4, False),
                                               ("pf", 1, 0, False), ("pf", 2, 3, False), ("pf", 2, 0, True),
                                               ("pf", 1, 4, True)])
def test_c_trajectory_equals_numpy_trajectory(kind, k, delay, cplx):
    """Same seeded inputs through both restatements: identical decisions, ratios and final
    state to rounding -- immediate and delayed (carriers, Eq. 10-15 / 25-28) alike."""
    seed, n, M, steps = 991 + k, 14, 30, 50
    if kind == "det":
        orb = wl.orbital_matrix(seed, 2, M, n, 1.0 / n, cplx)
    else:
        orb = wl.pairing_matrix(seed, 2, M, 1.0 / n, cplx)
    occ, unocc = wl.initial_occupation(seed, 2, M, n)
    P, J, xi = wl.proposals(seed, 3, steps, n, M, k, walkers=[2])
    a = getattr(pyorc, kind + "_trajectory")(orb, occ, unocc, P[:, 0], J[:, 0], xi[:, 0], scratch_every=3, delay=delay)
    b = getattr(c_oracle, kind + "_trajectory")(orb, occ, unocc, P[:, 0], J[:, 0], xi[:, 0], scratch_every=3, delay=delay)
    assert np.array_equal(a["accepted"], b["accepted"]) and a["accepted"].sum() > 3
    np.testing.assert_allclose(a["r_lemma"], b["r_lemma"], rtol=1e-8)
    m = ~np.isnan(a["r_scratch"])
    assert np.array_equal(m, ~np.isnan(b["r_scratch"]))
    np.testing.assert_allclose(a["r_scratch"][m], b["r_scratch"][m], rtol=1e-9)
    assert np.array_equal(a["occ"], b["occ"]) and np.array_equal(a["A"], b["A"])
    assert np.allclose(a["Ainv"], b["Ainv"], rtol=1e-7, atol=1e-9)
    assert a["logabs"] == pytest.approx(b["logabs"], abs=1e-9)
    assert a["scratch_logabs"] == pytest.approx(b["scratch_logabs"], abs=1e-10)
    assert a["phase"] == pytest.approx(b["phase"], abs=1e-9)
    assert a["init_logabs"] == pytest.approx(b["init_logabs"], abs=1e-11)


def test_c_batch_runs_walkers_independently():
    """orc_batch (OpenMP over walkers) gives each walker exactly its single-walker result,
    and scratch_every = 0 changes no tracked value (only the from-scratch checks go away)."""
    seed, W, n, M, k, steps = 555, 5, 12, 24, 2, 30
    orb = np.stack([wl.orbital_matrix(seed, w, M, n, 1.0 / n) for w in range(W)])
    occ, unocc = wl.initial_occupations(seed, W, M, n)
    P, J, xi = wl.proposals(seed, W, steps, n, M, k)
    res = c_oracle.batch("det", orb, occ, unocc, P, J, xi, scratch_every=1, threads=3)
    res0 = c_oracle.batch("det", orb, occ, unocc, P, J, xi, scratch_every=0, threads=2)
    for w in range(W):
        one = c_oracle.det_trajectory(orb[w], occ[w], unocc[w], P[:, w], J[:, w], xi[:, w])
        for key in ("r_lemma", "accepted", "occ", "Ainv"):
            assert np.array_equal(res[w][key], one[key]) and np.array_equal(res0[w][key], one[key])
        assert res[w]["logabs"] == one["logabs"] == res0[w]["logabs"]
        assert res0[w]["scratch_logabs"] == one["scratch_logabs"]
        assert np.isnan(res0[w]["r_scratch"]).all()
