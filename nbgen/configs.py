"""BASELINE.json configs 1-5 as seeded synthetic inputs (shapes only -- see nbgen/__init__.py).

``make_config(k, ...)`` returns a plain dict:

    name, N, cap, nb_target, t            scalars
    m, t0                [N]     float64
    x0, v0, a0, j0       [N,3]   float64   (a0/j0 are None for config 1 until the caller fills them)
    idx_i                [n_i]   int32     active block (unique, in range)
    h2_i                 [n_i]   float64   neighbour radius squared per active particle
                                           (None for config 1 until ``finish_config1``)
    order                [N]     int32     nested active-block order (configs 3-5): the first n
                                           entries are the active block of size n
    h2_all               [N]     float64   h^2 for every particle (configs 2-5) so that blocks of any
                                           size can be cut with ``active_block``

``N`` may be overridden to shrink a config for CPU-side tests; the recipe is unchanged.
"""
from __future__ import annotations

import numpy as np

from . import cluster as C

CONFIG_NAMES = {
    1: "cfg1_plummer1k_equal_all_active",
    2: "cfg2_plummer64k_kroupa_block4096",
    3: "cfg3_plummer256k_kroupa_bin5_sweep",
    4: "cfg4_plummer1m_kroupa_bin5_headline",
    5: "cfg5_king9_1m_core_overflow",
}

A_HENON = 3.0 * np.pi / 16.0        # Plummer scale with E = -1/4 (configs 1-3)
A_RH1 = 1.0 / 1.30477               # Plummer scale with half-mass radius 1 (config 4)


def _radius(x):
    return np.sqrt(np.einsum("ij,ij->i", x, x))


def _nested_order_by_level(levels, seed):
    """Active-block order for configs 3-4: deepest level first, ties by a seeded shuffle."""
    key = C.substream(seed, "block").random(levels.size)
    return np.lexsort((key, -levels.astype(np.int64))).astype(np.int32)


def active_block(cfg: dict, n_i: int):
    """Cut the nested active block of size n_i out of a config 3-5 dict."""
    idx = np.ascontiguousarray(cfg["order"][:n_i], dtype=np.int32)
    return idx, np.ascontiguousarray(cfg["h2_all"][idx])


def shard_active_block(idx_i: np.ndarray, h2_i: np.ndarray, rank: int, world: int):
    """i-sharding of one active block over ``world`` ranks (the paper's copy algorithm, P:59:
    every rank holds all j, ranks split the active set).  Contiguous, balanced, covers every
    element exactly once."""
    n = idx_i.shape[0]
    lo = (n * rank) // world
    hi = (n * (rank + 1)) // world
    return idx_i[lo:hi], h2_i[lo:hi]


def make_config(k: int, N: int | None = None, n_i: int | None = None, seed: int = 0) -> dict:
    if k == 1:
        N = N or 1024
        x, v = C.plummer_model(N, A_HENON, seed)
        m = np.full(N, 1.0 / N)
        x, v = C.center_of_mass_frame(m, x, v)
        return dict(name=CONFIG_NAMES[1], N=N, cap=256, nb_target=48, t=2.0 ** -10,
                    m=m, x0=x, v0=v, a0=None, j0=None, t0=np.zeros(N),
                    idx_i=np.arange(N, dtype=np.int32), h2_i=None, a_plummer=A_HENON)

    if k == 2:
        N = N or 65536
        a = A_HENON
        x, v = C.plummer_model(N, a, seed)
        m = C.kroupa_masses(N, seed)
        m /= m.sum()
        x, v = C.center_of_mass_frame(m, x, v)
        a0, j0 = C.plummer_smooth_field(x, v, a)
        lev = C.block_levels_uniform(N, 8, 14, seed)
        t = 1.0
        n_i = n_i or min(4096, N)
        idx = np.sort(C.substream(seed, "block").choice(N, size=n_i, replace=False)).astype(np.int32)
        h2_all = C.h2_from_density(C.plummer_number_density(_radius(x), N, a), 100.0)
        return dict(name=CONFIG_NAMES[2], N=N, cap=512, nb_target=100, t=t, m=m, x0=x, v0=v,
                    a0=a0, j0=j0, t0=C.t0_from_levels(lev, t), levels=lev,
                    idx_i=idx, h2_i=h2_all[idx].copy(), h2_all=h2_all, a_plummer=a)

    if k in (3, 4):
        N = N or (262144 if k == 3 else 1048576)
        a = A_HENON if k == 3 else A_RH1
        target = 100.0 if k == 3 else 150.0
        x, v = C.plummer_model(N, a, seed)
        m_sun = C.kroupa_masses(N, seed)
        m_sun, which, _semi = C.merge_binaries(m_sun, 0.05, seed)
        m = m_sun / m_sun.sum()
        x, v = C.center_of_mass_frame(m, x, v)
        a0, j0 = C.plummer_smooth_field(x, v, a)
        r = _radius(x)
        lev = C.block_levels_powerlaw(r, 8, 18, seed)
        t = 1.0
        order = _nested_order_by_level(lev, seed)
        h2_all = C.h2_from_density(C.plummer_number_density(r, N, a), target)
        cfg = dict(name=CONFIG_NAMES[k], N=N, cap=512, nb_target=int(target), t=t, m=m, x0=x, v0=v,
                   a0=a0, j0=j0, t0=C.t0_from_levels(lev, t), levels=lev, order=order,
                   h2_all=h2_all, binaries=which, a_plummer=a,
                   sweep=[256, 1024, 4096, 16384, 65536] if k == 3
                   else [2 ** p for p in range(6, 18)])
        n_i = n_i or min(4096 if k == 3 else 8192, N)
        cfg["idx_i"], cfg["h2_i"] = active_block(cfg, n_i)
        return cfg

    if k == 5:
        N = N or 1048576
        model = C.KingModel(9.0)
        x, v = C.king_sample(N, model, seed)
        heavy = C.substream(seed, "heavy").random(N) < 0.01
        m = np.where(heavy, 10.0, 1.0)
        m = m / m.sum()
        x, v = C.center_of_mass_frame(m, x, v)
        a0, j0 = model.smooth_field(x, v)
        r = _radius(x)
        lev = C.block_levels_powerlaw(r, 8, 18, seed)
        t = 1.0
        order = np.argsort(r, kind="stable").astype(np.int32)       # innermost first
        ndens = N * model.density(r)                                  # number density (mean mass 1/N)
        h2 = C.h2_from_density(ndens, 150.0)
        # floor: radius that holds ~floor_target bodies at the CENTRAL density, so the flat core sits
        # right at the 512 cap (Poisson scatter mixes overflowing / non-overflowing i); the 10x stars
        # get twice the radius (8x the count: deep overflow).  Constants recorded in the bench output.
        floor_target = 520.0
        h2_floor = float(C.h2_from_density(np.array([N * model.density(0.0)]), floor_target)[0])
        h2 = np.maximum(h2, h2_floor)
        h2 = np.where(heavy, 4.0 * h2, h2)
        cfg = dict(name=CONFIG_NAMES[5], N=N, cap=512, nb_target=150, t=t, m=m, x0=x, v0=v,
                   a0=a0, j0=j0, t0=C.t0_from_levels(lev, t), levels=lev, order=order, h2_all=h2,
                   heavy=heavy, h2_floor=h2_floor, floor_target=floor_target, sweep=[32, 128, 512],
                   king_r_core=model.r_core, king_r_tidal=model.r_tidal)
        n_i = n_i or min(512, N)
        cfg["idx_i"], cfg["h2_i"] = active_block(cfg, n_i)
        return cfg

    raise ValueError(f"unknown config {k}")


def finish_config1(cfg: dict, a0: np.ndarray, j0: np.ndarray, xp: np.ndarray) -> dict:
    """Config 1 needs two method results as INPUTS (BASELINE.json configs[0]): a0/j0 from a full
    direct sum at t0 and h_i^2 = (1.01 x distance to the 48th nearest neighbour at the PREDICTED
    positions)^2.  The caller computes a0, j0 and xp (in the tests: with the oracle) and passes
    them in; this function only does the KD-tree radius query."""
    cfg = dict(cfg)
    cfg["a0"], cfg["j0"] = a0, j0
    cfg["h2_i"] = C.knn_radius2(xp, int(cfg["nb_target"]), 1.01)
    return cfg
