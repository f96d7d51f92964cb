"""Pins of oracle/hermite_ac.py (two-level Ahmad-Cohen stepping, readings R33-R38) against what the
mathematics fixes: the two limits in which the scheme must BE the single-level Hermite integrator, energy
conservation, block invariants and force-polynomial consistency.  CPU only."""
import numpy as np
import pytest

import nbgen
from oracle import hermite as H
from oracle import hermite_ac as AC


def _direct_force(m, xp, vp, idx):
    import oracle
    out = oracle.regular(m, xp, vp, idx, np.zeros(idx.shape[0]), 8, want_list=False)
    return out["acc"], out["jerk"]


def _energy(oracle, m, x, v):
    N = m.shape[0]
    pot = oracle.regular(m, x, v, np.arange(N, dtype=np.int32), np.zeros(N), 8, want_list=False)["pot"]
    return 0.5 * (m * (v * v).sum(1)).sum() + 0.5 * (m * pot).sum()


def _radii(x, k):
    """h2 so that every body has about k neighbours: (1.001 x distance to its k-th nearest)^2."""
    d2 = ((x[:, None, :] - x[None, :, :]) ** 2).sum(-1)
    return np.sort(d2, axis=1)[:, k] * 1.002


def test_no_neighbours_is_the_single_level_integrator(oracle):
    """Every h2 = 0: no irregular force, dtI = dtR (R36), the irregular corrector adds nothing and the regular
    correction IS the Hermite corrector: same states (to the rounding of one regrouped sum), same steps,
    same blocks as oracle.hermite.integrate.  A wrong sign, a missing term or a wrong step in the regular
    branch breaks this."""
    N = 96
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    eta, eta_s, dt_max, t_end = 0.02, 0.02, 2.0**-4, 0.125
    ref = H.integrate(m, x, v, t_end, eta, eta_s, dt_max, _direct_force)
    st = AC.integrate(oracle, m, x, v, np.zeros(N), 8, t_end, eta_I=0.005, eta_R=eta, eta_s=eta_s, dt_max=dt_max)
    assert st["blocks"] == ref["blocks"] and st["regular_steps"] == ref["particle_steps"] == st["irregular_steps"]
    assert np.array_equal(st["dtR"], ref["dt"]) and np.array_equal(st["dtI"], st["dtR"])
    assert np.abs(st["x0"] - ref["x0"]).max() < 1e-13 and np.abs(st["v0"] - ref["v0"]).max() < 1e-12
    assert np.abs(st["a0"] - ref["a0"]).max() < 1e-11 * np.abs(ref["a0"]).max()
    assert not st["aI"].any() and st["nnb"].sum() == 0


def test_everybody_a_neighbour_is_the_single_level_integrator(oracle):
    """Every body inside every radius: no regular force, the irregular branch alone is the Hermite scheme with
    dt_max = dtR; the regular steps every dt_max are no-ops."""
    N = 48
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    eta, eta_s, dt_max, t_end = 0.02, 0.02, 2.0**-5, 0.0625
    ref = H.integrate(m, x, v, t_end, eta, eta_s, dt_max, _direct_force)
    st = AC.integrate(oracle, m, x, v, np.full(N, 1e6), N, t_end, eta_I=eta, eta_R=0.5, eta_s=eta_s, dt_max=dt_max)
    assert st["irregular_steps"] == ref["particle_steps"] and st["blocks"] == ref["blocks"]
    assert np.array_equal(st["dtI"], ref["dt"]) and np.all(st["dtR"] == dt_max)
    assert np.abs(st["x0"] - ref["x0"]).max() < 1e-13 and np.abs(st["v0"] - ref["v0"]).max() < 1e-12
    assert not st["aR"].any() and np.all(st["nnb"] == N - 1)


def test_two_level_run_conserves_energy_and_keeps_the_invariants(oracle):
    """Real radii (about 12 neighbours of 192 bodies): the energy error is at the level of the single-level run
    and falls with smaller eta; along the run dtI <= dtR, both are powers of 0.5, regular times are irregular
    times, t0 / tR are multiples of dtI / dtR, the stored total force is aI + aR + jR (t0 - tR), most steps are
    irregular, and for a body whose list did not change at a regular step the regular force w.r.t. the old
    list equals the one w.r.t. the new list."""
    N, cap = 192, 96
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    h2 = _radii(x, 12)
    eta_s, dt_max, t_end = 0.01, 2.0**-4, 0.25
    e0 = _energy(oracle, m, x, v)
    seen = dict(blocks=0, unchanged=0, changed=0)
    prev_lists = {}

    def on_block(t, act, reg, st):
        seen["blocks"] += 1
        assert np.all(st["dtI"] <= st["dtR"]) and np.all(st["tR"] <= st["t0"])
        for d in (st["dtI"], st["dtR"]):
            lev = -np.log2(d)
            assert np.all(lev == np.round(lev)) and d.max() <= dt_max
        assert np.all(st["t0"] / st["dtI"] == np.floor(st["t0"] / st["dtI"]))
        assert np.all(st["tR"] / st["dtR"] == np.floor(st["tR"] / st["dtR"]))
        nxt = (st["tR"] + st["dtR"]) / st["dtI"]
        assert np.all(nxt == np.floor(nxt))                              # the next regular time is an irregular time
        assert np.isin(reg, act).all()
        tot = st["aI"] + st["aR"] + st["jR"] * (st["t0"] - st["tR"])[:, None]
        assert np.abs(tot - st["a0"]).max() <= 1e-13 * np.abs(st["a0"]).max()
        if reg.size:
            ridx, aR1_old = st["_last_reg"]
            for q, i in enumerate(ridx):
                new = tuple(st["list"][i, :st["nnb"][i]])
                if prev_lists.get(int(i)) == new:
                    seen["unchanged"] += 1
                    assert np.abs(aR1_old[q] - st["aR"][i]).max() <= 1e-11 * max(np.abs(st["aR"][i]).max(), 1e-300)
                else:
                    seen["changed"] += 1
                prev_lists[int(i)] = new

    st = AC.integrate(oracle, m, x, v, h2, cap, t_end, eta_I=0.01, eta_R=0.02, eta_s=eta_s, dt_max=dt_max, on_block=on_block)
    assert np.all(st["t0"] == t_end) and np.all(st["tR"] == t_end)
    e1 = _energy(oracle, m, st["x0"], st["v0"])
    err = abs((e1 - e0) / e0)
    print("AC run: blocks", st["blocks"], "irregular steps", st["irregular_steps"], "regular steps", st["regular_steps"],
          "dE/E", err, "lists unchanged/changed at regular steps", seen["unchanged"], seen["changed"])
    assert st["irregular_steps"] > 2 * st["regular_steps"] > 0            # a real two-level run
    assert seen["unchanged"] > 0 and seen["changed"] > 0
    assert err < 2e-6
    st2 = AC.integrate(oracle, m, x, v, h2, cap, t_end, eta_I=0.0025, eta_R=0.005, eta_s=0.0025, dt_max=dt_max)
    e2 = _energy(oracle, m, st2["x0"], st2["v0"])
    assert abs((e2 - e0) / e0) < 0.5 * err + 1e-12
    # against the single-level run at the same accuracy parameter: same physics, positions agree to the
    # integration error of either (not a rounding-level identity)
    ref = H.integrate(m, x, v, t_end, 0.0025, 0.0025, dt_max, _direct_force)
    assert np.abs(st2["x0"] - ref["x0"]).max() < 1e-6


def test_overflow_is_an_error(oracle):
    N = 32
    cfg = nbgen.make_config(1, N=N)
    with pytest.raises(OverflowError):
        AC.start(oracle, cfg["m"], cfg["x0"], cfg["v0"], np.full(N, 1e6), 8, 0.01, 2.0**-4)


def test_irregular_step_never_exceeds_the_regular_step(oracle):
    """A regular criterion far stricter than the irregular one (eta_R << eta_I) makes dtR collapse at a regular
    step while the irregular criterion would keep dtI: the cap dtI <= dtR (R34/R35) must bite."""
    N, cap = 64, 48
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    h2 = _radii(x, 8)
    st = AC.start(oracle, m, x, v, h2, cap, 0.05, 2.0**-4)
    capped = 0
    for _ in range(12):
        before_I = st["dtI"].copy()
        t, act, reg = AC.block_step(oracle, m, st, h2, cap, eta_I=0.5, eta_R=1e-7, dt_max=2.0**-4)
        assert np.all(st["dtI"] <= st["dtR"])
        capped += int((st["dtI"][reg] < 0.5 * before_I[reg]).sum())          # pulled down by dtR, not by its own criterion
        nxt = (st["tR"] + st["dtR"]) / st["dtI"]
        assert np.all(nxt == np.floor(nxt))
    assert capped > 0
