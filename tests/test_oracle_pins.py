"""Pins for the CPU oracle (oracle/nbody_oracle.c) against things OTHER than itself:
closed forms, calculus identities checked by finite differences, conservation laws, a textbook
potential energy, a library KD-tree, exact rational arithmetic and a second brute-force written
a different way.  No GPU needed.  (north_star oracle checks; SURVEY.md 8(c) "What pins each part".)
"""
import math
from fractions import Fraction
from pathlib import Path

import numpy as np
import pytest
from scipy.spatial import cKDTree

import nbgen

GOLD = Path(__file__).parent / "golden"


def _rand_system(n, seed, spread=1.0):
    rng = np.random.default_rng(seed)
    x = rng.normal(size=(n, 3)) * spread
    v = rng.normal(size=(n, 3)) * 0.5
    m = rng.uniform(0.2, 1.0, size=n)
    m /= m.sum()
    return m, x, v


def _total(orc, m, x, v, idx=None):
    n = m.size
    idx = np.arange(n, dtype=np.int32) if idx is None else idx
    return orc.regular(m, x, v, idx, np.zeros(idx.size), cap=4)


# ----------------------------------------------------------------------------- pair formulas

def test_two_body_golden(oracle):
    rows = {}
    for line in (GOLD / "two_body.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            k, *vals = line.split()
            rows[k] = np.array([float(s) for s in vals])
    m = np.array([1.0, rows["m"][0]])
    x = np.stack([np.zeros(3), rows["r"]])
    v = np.stack([np.zeros(3), rows["v"]])
    out = oracle.regular(m, x, v, np.array([0], np.int32), np.array([0.0]), cap=4)
    np.testing.assert_allclose(out["acc"][0], rows["acc"], rtol=0, atol=1e-16)
    np.testing.assert_allclose(out["jerk"][0], rows["jerk"], rtol=0, atol=1e-16)
    assert abs(out["pot"][0] - rows["pot"][0]) < 1e-16
    assert out["nnb"][0] == 0 and out["overflow"][0] == 0
    # the partner sees the mirrored force scaled by the other mass (m_i = 1 here as well)
    out1 = oracle.regular(m, x, v, np.array([1], np.int32), np.array([0.0]), cap=4)
    np.testing.assert_allclose(out1["acc"][0], -rows["acc"], atol=1e-16)
    np.testing.assert_allclose(out1["jerk"][0], -rows["jerk"], atol=1e-16)


def test_circular_binary_closed_form(oracle):
    m = np.array([0.7, 0.3]); d = 0.37
    omega = math.sqrt(m.sum() / d ** 3)
    x = np.array([[-m[1] * d, 0, 0], [m[0] * d, 0, 0]]) / m.sum()
    v = np.array([[0, -m[1] * d * omega, 0], [0, m[0] * d * omega, 0]]) / m.sum()
    out = _total(oracle, m, x, v)
    a, j = out["acc"], out["jerk"]
    for i, other in ((0, 1), (1, 0)):
        assert abs(np.linalg.norm(a[i]) - m[other] / d ** 2) < 1e-14
        assert abs(np.dot(a[i], j[i])) < 1e-13 * np.linalg.norm(a[i]) * np.linalg.norm(j[i])
        assert abs(np.linalg.norm(j[i]) - omega * np.linalg.norm(a[i])) < 1e-13 * np.linalg.norm(j[i])
        assert abs(out["pot"][i] + m[other] / d) < 1e-15
    # jerk points along the partner's relative velocity direction (force vector rotates with omega)
    assert j[0][1] > 0 and abs(j[0][0]) < 1e-13


def test_jerk_is_time_derivative_of_acc_and_acc_is_minus_grad_pot(oracle):
    """Calculus pins: with every body moving on a straight line x(t) = x + v t (constant v),
    d/dt acc_i = jerk_i exactly; and acc_i = -d(pot_i)/d(x_i).  Central differences, O(eps^2)."""
    m, x, v = _rand_system(24, 1)
    base = _total(oracle, m, x, v)
    eps = 1e-5
    ap = _total(oracle, m, x + eps * v, v)["acc"]
    am = _total(oracle, m, x - eps * v, v)["acc"]
    fd_jerk = (ap - am) / (2 * eps)
    scale = np.linalg.norm(base["jerk"], axis=1, keepdims=True)
    assert np.max(np.abs(fd_jerk - base["jerk"]) / scale) < 2e-7
    for i in (0, 7, 23):
        for c in range(3):
            xs = x.copy(); xs[i, c] += eps
            pp = _total(oracle, m, xs, v, np.array([i], np.int32))["pot"][0]
            xs[i, c] -= 2 * eps
            pm = _total(oracle, m, xs, v, np.array([i], np.int32))["pot"][0]
            assert abs(-(pp - pm) / (2 * eps) - base["acc"][i, c]) < 1e-7 * np.linalg.norm(base["acc"][i])


def _brute_pairs(m, x, v, idx, h2):
    """Second, independent formulation: loop over UNORDERED pairs (Newton's third law), per-pair
    scalars via math.dist / pow, sums via math.fsum.  Returns per-particle totals and the
    neighbour partition by explicit set membership."""
    n = len(m)
    terms = [[[] for _ in range(7)] for _ in range(n)]       # total
    reg = [[[] for _ in range(7)] for _ in range(n)]
    nbs = [set() for _ in range(n)]
    h2full = {int(i): float(h) for i, h in zip(idx, h2)}
    for a in range(n):
        for b in range(a + 1, n):
            d = math.dist(x[a], x[b])
            rv = sum((x[b][c] - x[a][c]) * (v[b][c] - v[a][c]) for c in range(3))
            inv3 = math.pow(d, -3.0)
            inv5 = math.pow(d, -5.0)
            for (p, q, sgn) in ((a, b, 1.0), (b, a, -1.0)):   # p feels q
                t = []
                for c in range(3):
                    t.append(m[q] * sgn * (x[b][c] - x[a][c]) * inv3)
                for c in range(3):
                    t.append(m[q] * sgn * ((v[b][c] - v[a][c]) * inv3 - 3.0 * rv * (x[b][c] - x[a][c]) * inv5))
                t.append(-m[q] / d)
                isnb = p in h2full and d * d < h2full[p]
                if isnb:
                    nbs[p].add(q)
                for s in range(7):
                    terms[p][s].append(t[s])
                    if not isnb:
                        reg[p][s].append(t[s])
    tot = np.array([[math.fsum(terms[p][s]) for s in range(7)] for p in range(n)])
    rg = np.array([[math.fsum(reg[p][s]) for s in range(7)] for p in range(n)])
    return tot, rg, nbs


@pytest.mark.parametrize("n,seed", [(2, 0), (3, 1), (17, 2), (64, 3)])
def test_brute_force_small_n(oracle, n, seed):
    m, x, v = _rand_system(n, seed)
    idx = np.arange(n, dtype=np.int32)
    h2 = np.full(n, 0.8 ** 2)
    tot, rg, nbs = _brute_pairs(m, x, v, idx, h2)
    out = oracle.regular(m, x, v, idx, h2, cap=n)
    got = np.concatenate([out["acc"], out["jerk"], out["pot"][:, None]], axis=1)
    sc = np.abs(tot).max(axis=0) + 1e-300
    assert np.max(np.abs(got - rg) / sc) < 1e-13
    tot_orc = _total(oracle, m, x, v)
    got_t = np.concatenate([tot_orc["acc"], tot_orc["jerk"], tot_orc["pot"][:, None]], axis=1)
    assert np.max(np.abs(got_t - tot) / sc) < 1e-13
    for i in range(n):
        assert out["nnb"][i] == len(nbs[i])
        assert set(out["nblist"][i, :out["nnb"][i]].tolist()) == nbs[i]
        assert list(out["nblist"][i, :out["nnb"][i]]) == sorted(nbs[i])


# ----------------------------------------------------------------------------- full-sum invariants

def test_momentum_conservation_all_active(oracle):
    m, x, v = _rand_system(300, 5)
    out = _total(oracle, m, x, v)
    fa = (m[:, None] * out["acc"]).sum(0)
    fj = (m[:, None] * out["jerk"]).sum(0)
    assert np.abs(fa).max() < 1e-13 * np.abs(m[:, None] * out["acc"]).sum()
    assert np.abs(fj).max() < 1e-13 * np.abs(m[:, None] * out["jerk"]).sum()
    # pair symmetry of the potential energy: sum_i m_i phi_i = -2 sum_{i<j} m_i m_j / r_ij
    d = np.linalg.norm(x[:, None] - x[None], axis=2)
    iu = np.triu_indices(len(m), 1)
    W = -(m[:, None] * m[None])[iu] / d[iu]
    assert abs((m * out["pot"]).sum() - 2 * W.sum()) < 1e-13 * abs(W.sum())


def test_regular_plus_neighbours_is_total(oracle):
    cfg = nbgen.make_config(2, N=2048, n_i=256)
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    h2 = cfg["h2_i"] * 4.0
    reg = oracle.regular(cfg["m"], xp, vp, cfg["idx_i"], h2, cfg["cap"])
    tot = oracle.regular(cfg["m"], xp, vp, cfg["idx_i"], np.zeros_like(h2), cfg["cap"])
    assert reg["nnb"].sum() > 1000 and tot["nnb"].sum() == 0
    for key in ("acc", "jerk", "pot"):
        s = reg[key] + reg[key + "_nb"]
        sc = np.abs(tot[key]).max()
        assert np.max(np.abs(s - tot[key])) < 1e-13 * max(sc, np.abs(reg[key + "_nb"]).max())
        assert np.all(tot[key + "_nb"] == 0)


def test_translation_permutation_mass_linearity(oracle):
    m, x, v = _rand_system(200, 7)
    idx = np.arange(0, 200, 3, dtype=np.int32)
    h2 = np.full(idx.size, 0.3)
    base = oracle.regular(m, x, v, idx, h2, cap=64)
    shift = np.array([100.0, -50.0, 25.0])
    sh = oracle.regular(m, x + shift, v + np.array([3.0, -1.0, 2.0]), idx, h2, cap=64)
    for key, tol in (("acc", 1e-12), ("jerk", 1e-12), ("pot", 1e-12)):
        assert np.max(np.abs(sh[key] - base[key])) < tol * np.abs(base[key]).max()
    assert np.array_equal(sh["nnb"], base["nnb"])
    perm = np.random.default_rng(0).permutation(200)
    inv = np.argsort(perm)
    pm = oracle.regular(m[perm], x[perm], v[perm], inv[idx].astype(np.int32), h2, cap=64)
    for key in ("acc", "jerk", "pot"):
        assert np.max(np.abs(pm[key] - base[key])) < 1e-14 * np.abs(base[key]).max()
    for k in range(idx.size):
        assert set(perm[pm["nblist"][k, :pm["nnb"][k]]]) == set(base["nblist"][k, :base["nnb"][k]])
    dbl = oracle.regular(2.0 * m, x, v, idx, h2, cap=64)
    for key in ("acc", "jerk", "pot"):
        assert np.array_equal(dbl[key], 2.0 * base[key])


def test_plummer_potential_and_virial(oracle):
    """W = 1/2 sum m_i phi_i(h2=0) ~ -(3 pi/32) G M^2 / a = -1/2 for a = 3 pi/16; T ~ 1/4 (virial).
    The generator does not rescale to the measured energy, so this is independent of it."""
    n = 4096
    x, v = nbgen.plummer_model(n, nbgen.configs.A_HENON, seed=3)
    m = np.full(n, 1.0 / n)
    out = _total(oracle, m, x, v, np.arange(n, dtype=np.int32))
    W = 0.5 * (m * out["pot"]).sum()
    T = 0.5 * (m * (v ** 2).sum(1)).sum()
    assert abs(W + 0.5) < 0.03, W          # finite-N scatter ~ N^-1/2 ~ 1.6 %
    assert abs(T - 0.25) < 0.02, T
    # config 4's scale radius (half-mass radius 1): W = -(3 pi / 32) / a = -0.3843
    a4 = nbgen.configs.A_RH1
    x4, v4 = nbgen.plummer_model(n, a4, seed=4)
    W4 = 0.5 * (m * _total(oracle, m, x4, v4, np.arange(n, dtype=np.int32))["pot"]).sum()
    assert abs(W4 + 3 * math.pi / 32 / a4) < 0.03 * 0.3843 * 2
    assert abs(np.median(np.linalg.norm(x4, axis=1)) - 1.0) < 0.05


# ----------------------------------------------------------------------------- neighbour lists

def test_neighbour_sets_match_kdtree(oracle):
    cfg = nbgen.make_config(3, N=4096, n_i=512)
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    out = oracle.regular(cfg["m"], xp, vp, cfg["idx_i"], cfg["h2_i"], cfg["cap"])
    tree = cKDTree(xp)
    for k, i in enumerate(cfg["idx_i"]):
        ball = set(tree.query_ball_point(xp[i], math.sqrt(cfg["h2_i"][k]) * (1 - 1e-12))) - {int(i)}
        assert out["nnb"][k] == len(ball)
        assert set(out["nblist"][k, :out["nnb"][k]].tolist()) == ball
    assert 40 < out["nnb"].mean() < 250


def test_overflow_semantics_and_cap_invariance(oracle):
    m, x, v = _rand_system(50, 9)
    idx = np.arange(50, dtype=np.int32)
    h2 = np.full(50, 1.0)
    big = oracle.regular(m, x, v, idx, h2, cap=64)
    assert big["overflow"].sum() == 0 and big["nnb"].max() > 4
    for cap in (1, 2):
        o = oracle.regular(m, x, v, idx, h2, cap=cap)
        assert np.array_equal(o["nnb"], big["nnb"])                     # true count
        assert np.array_equal(o["overflow"], (big["nnb"] > cap).astype(np.int32))
        for key in ("acc", "jerk", "pot"):                              # force excludes ALL neighbours
            assert np.array_equal(o[key], big[key])
        for k in range(50):
            stored = o["nblist"][k, :min(cap, o["nnb"][k])]
            assert set(stored.tolist()) <= set(big["nblist"][k, :big["nnb"][k]].tolist())
            assert len(set(stored.tolist())) == min(cap, o["nnb"][k])


def test_nnb_monotone_symmetric_and_self_excluded(oracle):
    m, x, v = _rand_system(120, 11)
    idx = np.arange(120, dtype=np.int32)
    prev = np.zeros(120, np.int32)
    for h in (0.0, 0.1, 0.3, 0.9, 2.0, 1e3):
        o = oracle.regular(m, x, v, idx, np.full(120, h * h), cap=128)
        assert np.all(o["nnb"] >= prev)
        prev = o["nnb"]
        L = [set(o["nblist"][k, :o["nnb"][k]].tolist()) for k in range(120)]
        for i in range(120):
            assert i not in L[i]                                        # self excluded by index
            for j in L[i]:
                assert i in L[j]                                        # equal h  =>  symmetric
    assert np.all(prev == 119)                                          # huge h: everyone but self
    o = oracle.regular(m, x, v, idx, np.full(120, -1.0), cap=8)        # h2 <= 0: no neighbours
    assert o["nnb"].sum() == 0
    # with everyone a neighbour the regular part is exactly zero
    o = oracle.regular(m, x, v, idx, np.full(120, 1e6), cap=128)
    assert not o["acc"].any() and not o["jerk"].any() and not o["pot"].any()


def test_band_pairs_reported_with_terms(oracle):
    m = np.array([0.5, 0.25, 0.25])
    x = np.array([[0, 0, 0], [1.0, 0, 0], [0, 3.0, 0]])
    v = np.array([[0, 0, 0], [0, 0.5, 0], [0.1, 0, 0]])
    h2 = np.array([1.0 / (1 + 2e-6)])           # pair (0,1): r2 = 1 = h2 (1 + 2e-6): just outside
    bp = oracle.band_pairs(m, x, v, np.array([0], np.int32), h2, band=1e-5)
    assert bp["k"].tolist() == [0] and bp["j"].tolist() == [1] and bp["r2"][0] == 1.0
    np.testing.assert_allclose(bp["terms"][0], [0.25, 0, 0, 0, 0.125, 0, -0.25], atol=1e-16)
    assert oracle.band_pairs(m, x, v, np.array([0], np.int32), h2, band=1e-6)["k"].size == 0


# ----------------------------------------------------------------------------- predictor

def test_predictor_dyadic_is_exact(oracle):
    """x0, v0 dyadic, a0 = 2*dyadic, j0 = 6*dyadic, dt = 2^-k: every term is exactly representable,
    so the FP64 result must equal exact rational arithmetic bit for bit."""
    rng = np.random.default_rng(0)
    n = 64
    q = lambda s: rng.integers(-2 ** 12, 2 ** 12, size=s) / 2.0 ** 8
    x0, v0, a0, j0 = q((n, 3)), q((n, 3)), 2 * q((n, 3)), 6 * q((n, 3))
    k = rng.integers(3, 9, size=n)
    t = 1.0
    t0 = t - 2.0 ** -k
    xp, vp = oracle.predict(x0, v0, a0, j0, t0, t)
    for j in range(n):
        dt = Fraction(1, 2 ** int(k[j]))
        for c in range(3):
            X, V, A, J = (Fraction(float(z[j, c])) for z in (x0, v0, a0, j0))
            assert Fraction(float(xp[j, c])) == X + V * dt + A * dt ** 2 / 2 + J * dt ** 3 / 6
            assert Fraction(float(vp[j, c])) == V + A * dt + J * dt ** 2 / 2


def test_predictor_closed_forms_and_consistency(oracle):
    rng = np.random.default_rng(1)
    n = 32
    x0, v0, a0, j0 = (rng.normal(size=(n, 3)) for _ in range(4))
    t0 = rng.uniform(0, 0.5, n)
    # constant acceleration (j0 = 0): textbook kinematics
    xp, vp = oracle.predict(x0, v0, a0, 0 * j0, t0, 0.75)
    dt = (0.75 - t0)[:, None]
    np.testing.assert_allclose(xp, x0 + v0 * dt + 0.5 * a0 * dt * dt, rtol=1e-15, atol=1e-15)
    np.testing.assert_allclose(vp, v0 + a0 * dt, rtol=1e-15, atol=1e-15)
    # d xp/dt = vp and d vp/dt = a0 + j0 dt (catches a wrong 1/2 or 1/6)
    eps = 1e-4
    xa, va = oracle.predict(x0, v0, a0, j0, t0, 0.75 + eps)
    xb, vb = oracle.predict(x0, v0, a0, j0, t0, 0.75 - eps)
    xc, vc = oracle.predict(x0, v0, a0, j0, t0, 0.75)
    np.testing.assert_allclose((xa - xb) / (2 * eps), vc, rtol=0, atol=1e-7)
    np.testing.assert_allclose((va - vb) / (2 * eps), a0 + j0 * dt, rtol=0, atol=1e-7)
    # dt = 0 returns the state; backward prediction is the same polynomial
    x_, v_ = oracle.predict(x0, v0, a0, j0, np.full(n, 0.3), 0.3)
    assert np.array_equal(x_, x0) and np.array_equal(v_, v0)


# ----------------------------------------------------------------------------- config 1 construction

def test_config1_construction(oracle):
    cfg = nbgen.make_config(1)
    n = cfg["N"]
    tot = oracle.regular(cfg["m"], cfg["x0"], cfg["v0"], cfg["idx_i"], np.zeros(n), cfg["cap"])
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], tot["acc"], tot["jerk"], cfg["t0"], cfg["t"])
    cfg = nbgen.finish_config1(cfg, tot["acc"], tot["jerk"], xp)
    out = oracle.regular(cfg["m"], xp, vp, cfg["idx_i"], cfg["h2_i"], cfg["cap"])
    # radius x1.01 => ~3 % more volume => 48 + Poisson(~1.5) neighbours, never fewer than 48
    assert out["nnb"].min() >= 48 and out["nnb"].max() < 64 and 48 <= out["nnb"].mean() < 52
    assert out["overflow"].sum() == 0


# ----------------------------------------------------------------------------- neighbour (irregular) force

def _golden_rows():
    rows = {}
    for line in (GOLD / "two_body.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            k, *vals = line.split()
            rows[k] = np.array([float(s) for s in vals])
    return rows


def test_irregular_two_body_golden_with_prediction(oracle):
    """The paper-derived worked example (tests/golden/two_body.txt) reached THROUGH the predictor:
    the partner starts at t0 = 0 with exactly representable a0, j0 chosen so that at t = 1/2 it sits at
    r = (3,4,0) with v = (1,2,2) (all terms dyadic: no rounding)."""
    g = _golden_rows()
    dt = 0.5
    a0 = np.array([2.0, -4.0, 0.0]); j0 = np.array([6.0, 0.0, -12.0])
    v0 = g["v"] - a0 * dt - j0 * dt ** 2 / 2
    x0 = g["r"] - v0 * dt - a0 * dt ** 2 / 2 - j0 * dt ** 3 / 6
    z = np.zeros(3)
    st = dict(m=np.array([1.0, g["m"][0]]), x0=np.stack([z, x0]), v0=np.stack([z, v0]), a0=np.stack([z, a0]),
              j0=np.stack([z, j0]), t0=np.zeros(2))
    out = oracle.irregular(st["m"], st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], dt,
                           np.array([0], np.int32), np.array([1], np.int32), np.array([[1, -1]], np.int32), cap=2)
    np.testing.assert_allclose(out["acc"][0], g["acc"], rtol=0, atol=1e-16)
    np.testing.assert_allclose(out["jerk"][0], g["jerk"], rtol=0, atol=1e-16)
    assert abs(out["pot"][0] - g["pot"][0]) < 1e-16
    # empty list -> exact zeros; nnb above cap -> only the cap stored entries count
    out = oracle.irregular(st["m"], st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], dt,
                           np.array([0, 0], np.int32), np.array([0, 7], np.int32), np.array([[1], [1]], np.int32), cap=1)
    assert not out["acc"][0].any() and out["pot"][0] == 0
    np.testing.assert_allclose(out["acc"][1], g["acc"], atol=1e-16)


def test_irregular_brute_force_numpy(oracle):
    """Second, independent statement in numpy (vectorised over the list) with random lists, random
    individual t0 and a random time t."""
    rng = np.random.default_rng(5)
    N, n, cap = 60, 17, 12
    m, x0, v0 = _rand_system(N, 11)
    a0 = rng.normal(size=(N, 3)); j0 = rng.normal(size=(N, 3)); t0 = rng.uniform(0, 0.1, N); t = 0.17
    idx = rng.choice(N, n, replace=False).astype(np.int32)
    nnb = rng.integers(0, cap + 4, n).astype(np.int32)              # some rows "overflowed"
    lst = np.full((n, cap), -1, np.int32)
    for k in range(n):
        others = np.setdiff1d(np.arange(N), [idx[k]])
        c = min(nnb[k], cap)
        lst[k, :c] = rng.choice(others, c, replace=False)
    out = oracle.irregular(m, x0, v0, a0, j0, t0, t, idx, nnb, lst, cap)
    dt = (t - t0)[:, None]
    xp = x0 + v0 * dt + a0 * dt ** 2 / 2 + j0 * dt ** 3 / 6
    vp = v0 + a0 * dt + j0 * dt ** 2 / 2
    for k in range(n):
        js = lst[k, :min(nnb[k], cap)]
        r = xp[js] - xp[idx[k]]; v = vp[js] - vp[idx[k]]
        d = np.linalg.norm(r, axis=1)
        rv = np.einsum("ij,ij->i", r, v)
        a = (m[js, None] * r / d[:, None] ** 3).sum(0)
        jk = (m[js, None] * (v / d[:, None] ** 3 - 3 * rv[:, None] * r / d[:, None] ** 5)).sum(0)
        p = -(m[js] / d).sum()
        np.testing.assert_allclose(out["acc"][k], a, rtol=1e-12, atol=1e-14)
        np.testing.assert_allclose(out["jerk"][k], jk, rtol=1e-11, atol=1e-13)
        assert abs(out["pot"][k] - p) <= 1e-13 * max(abs(p), 1e-3)


def test_irregular_plus_regular_is_total(oracle):
    """regular = outside the neighbour radius, irregular = the neighbours.  With the lists the
    regular pass emits, irregular equals that pass's own neighbour sums and regular + irregular is the
    total direct force at the same time."""
    cfg = nbgen.make_config(2, N=2048, n_i=256)
    st = [cfg[k] for k in ("m", "x0", "v0", "a0", "j0", "t0")]
    xp, vp = oracle.predict(*st[1:], cfg["t"])
    h2 = cfg["h2_i"] * 4.0
    cap = 2048
    reg = oracle.regular(cfg["m"], xp, vp, cfg["idx_i"], h2, cap)
    tot = oracle.regular(cfg["m"], xp, vp, cfg["idx_i"], np.zeros_like(h2), cap)
    irr = oracle.irregular(*st, cfg["t"], cfg["idx_i"], reg["nnb"], reg["nblist"], cap)
    assert reg["overflow"].sum() == 0 and reg["nnb"].sum() > 1000
    for key in ("acc", "jerk", "pot"):
        sc = np.abs(reg[key + "_nb"]).max()
        assert np.max(np.abs(irr[key] - reg[key + "_nb"])) < 1e-13 * sc
        assert np.max(np.abs(reg[key] + irr[key] - tot[key])) < 1e-13 * max(sc, np.abs(tot[key]).max())
