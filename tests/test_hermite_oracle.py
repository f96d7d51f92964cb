"""Pins of oracle/hermite.py (block selection, Hermite corrector, block time step)
against what the mathematics fixes -- none of them re-types the oracle's own formulas."""
from fractions import Fraction

import numpy as np

import nbgen
from oracle import hermite as H


# ----------------------------------------------------------------------------- corrector

def _cubic_motion(c, x0, v0, t):
    """Exact x(t), v(t), a(t), j(t) for an acceleration a(t) = c0 + c1 t + c2 t^2 + c3 t^3 (Fractions)."""
    a = c[0] + c[1] * t + c[2] * t**2 + c[3] * t**3
    j = c[1] + 2 * c[2] * t + 3 * c[3] * t**2
    v = v0 + c[0] * t + c[1] * t**2 / 2 + c[2] * t**3 / 3 + c[3] * t**4 / 4
    x = x0 + v0 * t + c[0] * t**2 / 2 + c[1] * t**3 / 6 + c[2] * t**4 / 12 + c[3] * t**5 / 20
    return x, v, a, j


def test_corrector_is_exact_for_a_cubic_acceleration():
    """The Hermite corrector integrates the cubic interpolant of the acceleration: when the true
    acceleration IS a cubic in t the corrected x, v are the exact ones and a2, a3 are its derivatives."""
    rng = np.random.default_rng(3)
    fr = lambda: Fraction(int(rng.integers(-64, 65)), 16)
    n = 5
    dts = [Fraction(1, 2**k) for k in (1, 3, 4, 6, 2)]
    rows = []
    for k in range(n):
        comp = []
        for _ in range(3):
            c = [fr(), fr(), fr(), fr()]
            x0, v0 = fr(), fr()
            x1, v1, a1, j1 = _cubic_motion(c, x0, v0, dts[k])
            comp.append((c, x0, v0, x1, v1, a1, j1))
        rows.append(comp)
    f = lambda sel: np.array([[float(sel(rows[k][d])) for d in range(3)] for k in range(n)])
    x1, v1, a2, a3 = H.correct(f(lambda r: r[1]), f(lambda r: r[2]), f(lambda r: r[0][0]), f(lambda r: r[0][1]),
                               np.array([float(d) for d in dts]), f(lambda r: r[5]), f(lambda r: r[6]))
    assert np.allclose(x1, f(lambda r: r[3]), rtol=0, atol=1e-12)
    assert np.allclose(v1, f(lambda r: r[4]), rtol=0, atol=1e-12)
    assert np.allclose(a2, f(lambda r: 2 * r[0][2]), rtol=0, atol=1e-9)
    assert np.allclose(a3, f(lambda r: 6 * r[0][3]), rtol=0, atol=1e-8)


def _kepler_energy_error(nsteps):
    """Two bodies on a circular orbit (m = 1/2 each, separation 1, G = 1: period 2 pi), one period with
    a shared step through predict -> force -> correct; returns |dE / E|."""
    m = np.array([0.5, 0.5])
    x = np.array([[0.5, 0, 0], [-0.5, 0, 0]], dtype=float)
    vc = 0.5 * np.sqrt(1.0)            # each body moves on radius 1/2 with omega = 1
    v = np.array([[0, vc, 0], [0, -vc, 0]], dtype=float)

    def force(x, v):                    # textbook two-body acceleration and jerk, written out here
        r = x[1] - x[0]; u = v[1] - v[0]
        r2 = r @ r; r3 = r2**1.5
        a = r / r3; jk = u / r3 - 3 * (r @ u) * r / (r2 * r3)
        return np.array([m[1] * a, -m[0] * a]), np.array([m[1] * jk, -m[0] * jk])

    def energy(x, v):
        return 0.5 * (m * (v * v).sum(1)).sum() - m[0] * m[1] / np.linalg.norm(x[1] - x[0])

    e0 = energy(x, v)
    dt = 2 * np.pi / nsteps
    a, jk = force(x, v)
    for _ in range(nsteps):
        xp = x + v * dt + a * dt**2 / 2 + jk * dt**3 / 6
        vp = v + a * dt + jk * dt**2 / 2
        a1, j1 = force(xp, vp)
        x, v, _, _ = H.correct(x, v, a, jk, np.full(2, dt), a1, j1)
        a, jk = a1, j1
    return abs((energy(x, v) - e0) / e0)


def test_corrector_is_fourth_order_on_a_kepler_orbit():
    e1, e2, e3 = _kepler_energy_error(64), _kepler_energy_error(128), _kepler_energy_error(256)
    assert e1 < 1e-4
    assert 12.0 < e1 / e2 < 40.0 and 12.0 < e2 / e3 < 40.0     # error ~ dt^4 (per period: 16x per halving, or better)


# ----------------------------------------------------------------------------- block selection and steps

def test_active_set_is_the_prefix_of_the_sorted_list():
    """P:89 / Figures 1-2: with block steps the active particles are the head of the step-sorted list."""
    rng = np.random.default_rng(5)
    N = 5000
    lev = rng.integers(3, 12, size=N)
    dt = 2.0 ** -lev.astype(float)
    for t_now in (0.0, 0.375, 1.0 - 2.0**-11, 2.0**-11 * 37):
        t0 = np.floor(t_now / dt) * dt                       # last block time of every particle: multiple of dt
        t_next, act = H.next_block(t0, dt)
        assert t_next == t_now + 2.0**-11 or t_next > t_now
        assert np.array_equal(act, H.sorted_list_prefix(dt, t_next))
        assert act.size >= (lev == 11).sum()


def test_quantize_step_rules():
    q = H.quantize_step
    d = 2.0**-6
    assert q([10.0], [d], 4 * d, 1.0)[0] == 2 * d             # may double at a commensurate time ...
    assert q([10.0], [d], 3 * d, 1.0)[0] == d                 # ... not at an odd multiple
    assert q([10.0], [d], 4 * d, d)[0] == d                   # never above dt_max
    assert q([1.5 * d], [d], 4 * d, 1.0)[0] == d              # needs a full factor of two to grow
    assert q([0.9 * d], [d], 4 * d, 1.0)[0] == d / 2
    assert q([0.2 * d], [d], 4 * d, 1.0)[0] == d / 8          # halves as often as needed
    assert H.initial_step(np.array([[1.0, 0, 0]]), np.array([[0, 3.0, 0]]), 0.03, 0.125)[0] == 2.0**-7


def _direct_force(m, xp, vp, idx):
    """Total force on the active block (the C oracle's direct sum, h2 = 0)."""
    import oracle
    out = oracle.regular(m, xp, vp, idx, np.zeros(idx.shape[0]), 8)
    return out["acc"], out["jerk"]


def test_block_step_integration_conserves_energy_and_keeps_the_block_invariants():
    import oracle
    N = 128
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]

    def energy(x, v):
        pot = oracle.regular(m, x, v, np.arange(N, dtype=np.int32), np.zeros(N), 8)["pot"]
        return 0.5 * (m * (v * v).sum(1)).sum() + 0.5 * (m * pot).sum()

    seen = []

    def force(m_, xp, vp, idx):
        seen.append(idx.shape[0])
        return _direct_force(m_, xp, vp, idx)

    e0 = energy(x, v)
    st = H.integrate(m, x, v, t_end=0.25, eta=0.01, eta_s=0.01, dt_max=2.0**-4, force=force)
    assert np.all(st["t0"] == 0.25)                                     # everyone synchronised at t_end
    lev = -np.log2(st["dt"])
    assert np.all(lev == np.round(lev)) and st["dt"].max() <= 2.0**-4   # powers of 0.5
    assert np.all(st["t0"] / st["dt"] == np.floor(st["t0"] / st["dt"]))
    assert st["blocks"] > 16 and st["particle_steps"] > 4 * N and min(seen[1:]) < N   # real block structure
    e1 = energy(st["x0"], st["v0"])
    assert abs((e1 - e0) / e0) < 2e-6
    # halving eta lowers the error (fourth-order scheme with an adaptive step): at least 2x better
    st2 = H.integrate(m, x, v, t_end=0.25, eta=0.0025, eta_s=0.0025, dt_max=2.0**-4, force=_direct_force)
    e2 = energy(st2["x0"], st2["v0"])
    assert abs((e2 - e0) / e0) < 0.5 * abs((e1 - e0) / e0) + 1e-12


# ----------------------------------------------------------------------------- time-step criterion (DESIGN R28)

def _harmonic(A, w, ph, e):
    """a(t) = A cos(phi) e and its first three time derivatives at phase phi = w t (closed forms)."""
    e = np.asarray(e, dtype=float) / np.linalg.norm(e)
    a = A * np.cos(ph) * e
    j = -A * w * np.sin(ph) * e
    a2 = -A * w * w * np.cos(ph) * e
    a3 = A * w**3 * np.sin(ph) * e
    return a, j, a2, a3


def test_aarseth_step_is_sqrt_eta_over_omega_for_harmonic_motion():
    """For a(t) = A cos(wt) e the products in Aarseth's criterion are |a||a2| + |j|^2 = A^2 w^2 and
    |j||a3| + |a2|^2 = A^2 w^4 at EVERY phase, so dt_req = sqrt(eta) / w exactly -- independent of A and
    of the phase.  A missing sqrt, a wrong power, swapped products or a2 not advanced to the end of the
    step (it is handed in at the START of the step: a2_0 = a2(t1) - dt a3) all break the constancy."""
    rows = []
    for A, w, eta in ((1.0, 1.0, 0.02), (3.5, 7.0, 0.01), (0.02, 0.25, 0.04), (40.0, 31.0, 0.0025)):
        for ph in (0.0, 0.3, 0.5 * np.pi, 1.1, 2.0, 3.0, 4.4, 6.0):
            for dt in (0.5, 2.0**-5):
                a, j, a2, a3 = _harmonic(A, w, ph, (1.0, -2.0, 0.5))
                rows.append((a, j, a2 - dt * a3, a3, dt, eta, np.sqrt(eta) / w))
    col = lambda q: np.array([r[q] for r in rows])
    for eta in sorted({r[5] for r in rows}):
        sel = col(5) == eta
        got = H.aarseth_step(col(0)[sel], col(1)[sel], col(2)[sel], col(3)[sel], col(4)[sel], eta)
        np.testing.assert_allclose(got, col(6)[sel], rtol=1e-12, atol=0)


def test_aarseth_step_hand_case_with_a2_advanced_to_the_end_of_the_step():
    """Worked by hand from the formula DESIGN R28 cites (Aarseth 1985; Makino & Aarseth 1992):
        dt_req = sqrt( eta (|a||a2| + |j|^2) / (|j||a3| + |a2|^2) ),   a2 = a2(t0) + dt a3.
    a1 = (0,0,3): |a| = 3;  j1 = (4,0,0): |j| = 4;  a3 = (1.5,0,0): |a3| = 1.5;  dt = 2;
    a2(t0) = (-3,3,4)  ->  a2 at the end = (-3,3,4) + 2 (1.5,0,0) = (0,3,4): |a2| = 5.
    numerator   = 3*5 + 4^2  = 31;   denominator = 4*1.5 + 5^2 = 31;   eta = 1/16  ->  dt_req = 1/4 exactly.
    With a2 taken at the START (|a2|^2 = 34) the value is sqrt((3 sqrt(34) + 16) / (16 * 40)) = 0.2287...;
    with the two products swapped it is sqrt((6 + 16) / (16 * (15 + 25))) = 0.1854...
    Second row, unequal norms everywhere: a1 = (2,3,6) (7), j1 = (1,2,2) (3), a3 = (0,0,2) (2), dt = 1/2,
    a2(t0) = (4,4,6) -> (4,4,7) (9): numerator 7*9 + 9 = 72, denominator 3*2 + 81 = 87, eta = 0.02:
    dt_req = sqrt(0.02 * 72 / 87) = sqrt(1.44 / 87) = 1.2 / sqrt(87) = 0.128653504..."""
    a1 = np.array([[0.0, 0.0, 3.0], [2.0, 3.0, 6.0]])
    j1 = np.array([[4.0, 0.0, 0.0], [1.0, 2.0, 2.0]])
    a2_0 = np.array([[-3.0, 3.0, 4.0], [4.0, 4.0, 6.0]])
    a3 = np.array([[1.5, 0.0, 0.0], [0.0, 0.0, 2.0]])
    dt = np.array([2.0, 0.5])
    assert H.aarseth_step(a1[:1], j1[:1], a2_0[:1], a3[:1], dt[:1], 1.0 / 16.0)[0] == 0.25
    got = H.aarseth_step(a1[1:], j1[1:], a2_0[1:], a3[1:], dt[1:], 0.02)[0]
    assert abs(got - 0.128653504180535) < 1e-14              # 1.2 / sqrt(87) = 1.2 / 9.327379053088816


def test_initial_step_hand_cases():
    """dt = largest power of 0.5 not above min(eta_s |a| / |j|, dt_max), by hand:
    |a| = 5, |j| = 2, eta_s = 0.02 -> 0.05 -> 2^-5 (0.03125 <= 0.05 < 0.0625); capped by dt_max = 2^-6;
    |a| = 1, |j| = 4, eta_s = 1 -> exactly 2^-2 stays 2^-2 (floor of an exact power);
    |a| = 13, |j| = 1, eta_s = 0.01 -> 0.13 -> 2^-3."""
    a = np.array([[3.0, 4.0, 0.0], [3.0, 4.0, 0.0], [0.0, 1.0, 0.0], [3.0, 4.0, 12.0]])
    j = np.array([[0.0, 0.0, 2.0], [0.0, 0.0, 2.0], [0.0, 0.0, 4.0], [1.0, 0.0, 0.0]])
    assert H.initial_step(a[:1], j[:1], 0.02, 1.0)[0] == 2.0**-5
    assert H.initial_step(a[1:2], j[1:2], 0.02, 2.0**-6)[0] == 2.0**-6
    assert H.initial_step(a[2:3], j[2:3], 1.0, 1.0)[0] == 2.0**-2
    assert H.initial_step(a[3:], j[3:], 0.01, 1.0)[0] == 2.0**-3


def test_degenerate_step_criterion_keeps_the_step_and_has_a_floor():
    """DESIGN.md reading R32 (the paper is silent): dt_req = 0 or NaN keeps the step instead of
    halving for ever; halving stops at dt_max 2^-40; start-up steps are clipped to [dt_max 2^-40, dt_max] and
    |a| = |j| = 0 gives dt_max.  All by hand."""
    q = H.quantize_step
    d = 2.0**-6
    assert q([0.0], [d], 4 * d, 1.0)[0] == d                       # no information: keep
    assert q([np.nan], [d], 4 * d, 1.0)[0] == d
    assert q([np.inf], [d], 4 * d, 1.0)[0] == 2 * d                # constant force: may grow as usual
    assert q([1e-300], [d], 4 * d, 1.0)[0] == 2.0**-40             # floor = dt_max 2^-40
    assert q([1e-300], [d], 4 * d, 2.0**-3)[0] == 2.0**-43
    assert q([1e-300], [d], 4 * d, 1.0, dt_min=2.0**-10)[0] == 2.0**-10
    # isolated body feeling nothing: a1 = j1 = 0 with non-zero old derivatives -> criterion 0 -> step kept
    z = np.zeros((1, 3))
    req = H.aarseth_step(z, z, np.array([[1.0, 0, 0]]), np.array([[0, 2.0, 0]]), np.array([d]), 0.02)
    assert req[0] == 0.0 and q(req, [d], 4 * d, 1.0)[0] == d
    one = np.array([[1.0, 0.0, 0.0]])
    assert H.initial_step(z, one, 0.02, 0.125)[0] == 0.125 * 2.0**-40      # |a| = 0: the floor
    assert H.initial_step(one, z, 0.02, 0.125)[0] == 0.125                 # |j| = 0: dt_max
    assert H.initial_step(z, z, 0.02, 0.125)[0] == 0.125                   # nothing known: dt_max
