"""Pins for the seeded input generators (nbgen/): they are not the method, but configs 3-5 rest on them (round-2
verdict, "What's missing" 2).  Each check is against something the generator does not compute itself: SURVEY.md
section 8(c) reading 21's check values for the IMF, numerical integration of the stated density / pdf, King's (1966)
tabulated concentration, the oracle's potential sum and the virial theorem, and the stated occupancy law of the block
levels (SURVEY 8(d) recipe; "deep blocks hold few particles")."""
import math

import numpy as np
import pytest
from scipy import integrate

import nbgen
from nbgen import cluster as C


def _kroupa_pdf(m):                          # unnormalised, continuous at 0.5 (SURVEY 8(c) reading 21)
    return np.where(m < 0.5, m ** -1.3, 0.5 ** (2.3 - 1.3) * m ** -2.3)


def test_kroupa_imf_fraction_mean_and_cdf():
    n = 200_000
    m = C.kroupa_masses(n, seed=1)
    assert m.min() >= 0.08 and m.max() <= 100.0
    # SURVEY.md:341 check values: fraction below 0.5 Msun = 0.7607, mean mass 0.574 Msun
    assert abs((m < 0.5).mean() - 0.7607) < 3.5 * math.sqrt(0.7607 * 0.2393 / n)
    assert abs(m.mean() - 0.574) < 0.02          # sigma_m ~ 1.9 (heavy tail) -> 0.004 on the mean
    # empirical CDF against quadrature of the stated pdf
    norm = integrate.quad(_kroupa_pdf, 0.08, 0.5)[0] + integrate.quad(_kroupa_pdf, 0.5, 100.0)[0]
    for q in (0.1, 0.2, 0.5, 1.0, 3.0, 10.0, 50.0):
        pts = [p for p in (0.5,) if 0.08 < p < q]
        cdf = integrate.quad(_kroupa_pdf, 0.08, q, points=pts or None)[0] / norm
        assert abs((m < q).mean() - cdf) < 4.0 * math.sqrt(max(cdf * (1 - cdf), 1e-6) / n), q
    assert abs(integrate.quad(_kroupa_pdf, 0.08, 0.5)[0] / norm - 0.7607) < 5e-4      # the survey's number itself
    # seeded: same stream, same masses; another stream, other masses
    assert np.array_equal(m, C.kroupa_masses(n, seed=1)) and not np.array_equal(m, C.kroupa_masses(n, seed=2))


def test_binaries_are_merged_into_centre_of_mass_bodies():
    n = 40_000
    m = C.kroupa_masses(n, seed=3)
    mb, which, semi = C.merge_binaries(m, 0.05, seed=3)
    assert which.size == math.floor(0.05 * n) and np.unique(which).size == which.size
    rest = np.setdiff1d(np.arange(n), which)
    assert np.array_equal(mb[rest], m[rest])                       # singles untouched
    comp = mb[which] - m[which]
    assert comp.min() >= 0.08 - 1e-12 and comp.max() <= 100.0      # the companion is an IMF draw of its own
    assert abs(comp.mean() - 0.574) < 0.1
    assert semi.min() >= 1e-5 and semi.max() <= 1e-2
    cfg = nbgen.make_config(3, N=8192, n_i=64)
    assert abs(cfg["m"].sum() - 1.0) < 1e-12 and cfg["binaries"].size == math.floor(0.05 * 8192)


def test_king_w0_9_structure():
    k = C.KingModel(9.0)
    # King (1966) / Binney & Tremaine table: W0 = 9 -> c = log10(r_t / r_0) = 2.12
    assert abs(math.log10(k.r_tidal / k.r_core) - 2.12) < 0.01
    assert abs(math.log10(C.KingModel(6.0).rt_model) - 1.255) < 0.01           # W0 = 6 (the paper's own): c = 1.25-1.26
    # the tabulated mass profile is the integral of the tabulated density
    r, rho = k.r, k.rho
    shell = integrate.cumulative_trapezoid(4.0 * np.pi * r * r * rho, r, initial=0.0)
    assert abs(shell[-1] - 1.0) < 2e-3
    assert np.abs(shell - k.Mfrac).max() < 3e-3
    assert k.W[0] == 9.0 and k.W[-1] == 0.0 and np.all(np.diff(k.W) <= 0)
    # a W0 = 9 model is centrally concentrated: the density has fallen by > 100 at ten King radii
    assert k.rho[0] > 100.0 * k.density(k.r_core * 10)


def test_king_sample_energy_and_virial(oracle):
    """N = 4096 bodies drawn from the W0 = 9 model: W_pot = -1/2 from the ORACLE's potential sum (not from the model's
    table), T = 1/4 (virial), both within finite-N scatter; radii follow the tabulated M(r)."""
    n = 4096
    model = C.KingModel(9.0)
    x, v = C.king_sample(n, model, seed=5)
    m = np.full(n, 1.0 / n)
    pot = oracle.regular(m, x, v, np.arange(n, dtype=np.int32), np.zeros(n), cap=4)["pot"]
    W = 0.5 * (m * pot).sum()
    T = 0.5 * (m * (v ** 2).sum(1)).sum()
    assert abs(W + 0.5) < 0.04, W            # a W0 = 9 core holds few bodies at N = 4096: scatter ~ 4 %
    assert abs(T - 0.25) < 0.02, T
    assert abs(2 * T + W) < 0.05
    r = np.linalg.norm(x, axis=1)
    assert r.max() <= model.r_tidal * (1 + 1e-9)
    for q in (0.1, 0.5, 0.9):
        rq = np.interp(q, model.Mfrac, model.r)
        assert abs((r < rq).mean() - q) < 4.0 * math.sqrt(q * (1 - q) / n)
    # isotropy of both vectors
    assert np.abs(x.mean(0)).max() < 4 * r.std() / math.sqrt(n) and np.abs((v / np.linalg.norm(v, axis=1)[:, None]).mean(0)).max() < 0.04
    # nobody is unbound: v^2 / 2 < W(r) sigma^2
    assert np.all(0.5 * (v ** 2).sum(1) <= model.W_of_r(r) * model.vel_scale ** 2 * (1 + 1e-9))


def test_block_levels_follow_the_halving_law_and_sit_deepest_at_the_centre():
    n = 262_144
    rng = np.random.default_rng(0)
    radius = rng.random(n) ** (1.0 / 3.0)
    lev = C.block_levels_powerlaw(radius, 8, 18, seed=0)
    assert lev.min() == 8 and lev.max() == 18
    cnt = np.bincount(lev, minlength=19)[8:]
    # population of level k ~ 2^-(k-8) (SURVEY.md:382); the +-1 jitter (1/4 each way) maps a halving law onto itself
    for k in range(1, 7):                    # interior levels with > 1000 bodies
        assert abs(cnt[k + 1] / cnt[k] - 0.5) < 0.05, (k, cnt)
    assert cnt[0] > 0.4 * n
    med = [np.median(radius[lev == k]) for k in range(8, 17)]
    assert all(a > b for a, b in zip(med, med[1:]))               # deeper level, smaller radius
    t0 = C.t0_from_levels(lev, 1.0)
    assert np.array_equal(t0 + 2.0 ** -lev.astype(float), np.ones(n))     # every level is due at t = 1 exactly
    u = C.block_levels_uniform(70_000, 8, 14, seed=0)
    assert np.abs(np.bincount(u)[8:] / 70_000 - 1 / 7).max() < 0.01
