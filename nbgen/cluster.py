"""Seeded samplers for the synthetic star clusters (inputs only; see nbgen/__init__.py).

Units: N-body (Henon) units, G = 1, total mass 1.  Everything is FP64.
Recipes: SURVEY.md section 8(d) table "Synthetic inputs"; DESIGN.md section "Input recipe".
"""
from __future__ import annotations

import numpy as np
from scipy.integrate import solve_ivp
from scipy.spatial import cKDTree
from scipy.special import erf

# One Philox key per (seed, piece): changing how one piece is drawn never shifts another.
STREAMS = {
    "pos": 1, "vel": 2, "mass": 3, "binary": 4, "level": 5, "block": 6, "heavy": 7,
    "jitter": 8, "dir": 9, "vdir": 10,
}


def substream(seed: int, name: str) -> np.random.Generator:
    key = np.array([np.uint64(seed), np.uint64(STREAMS[name])], dtype=np.uint64)
    return np.random.Generator(np.random.Philox(key=key))


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    z = 1.0 - 2.0 * rng.random(n)
    phi = 2.0 * np.pi * rng.random(n)
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


# --------------------------------------------------------------------------- Plummer

def plummer_positions(n: int, a: float, seed: int, rmax_over_a: float = 25.0) -> np.ndarray:
    """Plummer sphere of scale radius ``a``: enclosed-mass fraction X in (0,1),
    r = a (X^(-2/3) - 1)^(-1/2), radii beyond ``rmax_over_a * a`` rejected."""
    rng = substream(seed, "pos")
    out = np.empty(0)
    while out.size < n:
        X = rng.random(n + n // 16 + 16)
        X = X[X > 0.0]
        r = a / np.sqrt(X ** (-2.0 / 3.0) - 1.0)
        out = np.concatenate([out, r[r <= rmax_over_a * a]])
    r = out[:n]
    return r[:, None] * _isotropic(substream(seed, "dir"), n)


def plummer_velocities(x: np.ndarray, a: float, seed: int, M: float = 1.0) -> np.ndarray:
    """Isotropic Plummer DF: q = v / v_esc drawn from g(q) ~ q^2 (1-q^2)^(7/2) by von Neumann
    rejection; v_esc = sqrt(2 G M / a) (1 + r^2/a^2)^(-1/4)."""
    n = x.shape[0]
    rng = substream(seed, "vel")
    q = np.zeros(n)
    pending = np.arange(n)
    while pending.size:
        x1 = rng.random(pending.size)
        x2 = rng.random(pending.size)
        ok = 0.1 * x2 < x1 * x1 * (1.0 - x1 * x1) ** 3.5
        q[pending[ok]] = x1[ok]
        pending = pending[~ok]
    r2 = np.einsum("ij,ij->i", x, x)
    vesc = np.sqrt(2.0 * M / a) * (1.0 + r2 / (a * a)) ** (-0.25)
    return (q * vesc)[:, None] * _isotropic(substream(seed, "vdir"), n)


def center_of_mass_frame(m, x, v):
    """Subtract the mass-weighted centre-of-mass position and velocity (no energy rescale, so
    that the Plummer potential-energy pin stays independent of the generator)."""
    mt = m.sum()
    return x - (m[:, None] * x).sum(0) / mt, v - (m[:, None] * v).sum(0) / mt


def plummer_model(n: int, a: float, seed: int):
    x = plummer_positions(n, a, seed)
    v = plummer_velocities(x, a, seed)
    return x, v


def plummer_smooth_field(x, v, a: float, M: float = 1.0):
    """a0, j0 of the SMOOTH Plummer model (O(N) stand-in for a full direct sum at N >= 65536,
    SURVEY 8(d) 'a0, j0'): a0 = -M x / (r^2+a^2)^(3/2), j0 = its convective derivative along v."""
    r2 = np.einsum("ij,ij->i", x, x) + a * a
    xv = np.einsum("ij,ij->i", x, v)
    i3 = r2 ** -1.5
    a0 = -M * x * i3[:, None]
    j0 = -M * (v * i3[:, None] - 3.0 * (xv * i3 / r2)[:, None] * x)
    return a0, j0


def plummer_number_density(r, n: int, a: float):
    return (3.0 * n / (4.0 * np.pi * a ** 3)) * (1.0 + (r / a) ** 2) ** (-2.5)


# --------------------------------------------------------------------------- masses

def kroupa_masses(n: int, seed: int, m_lo: float = 0.08, m_br: float = 0.5, m_hi: float = 100.0,
                  stream: str = "mass") -> np.ndarray:
    """Two-segment Kroupa (2001) IMF, dN/dm ~ m^-1.3 on [m_lo, m_br), ~ m^-2.3 on [m_br, m_hi],
    continuous at m_br; inverse-CDF sampling.  Returns masses in solar units (NOT normalised)."""
    a1, a2 = 1.3, 2.3
    # unnormalised segment integrals with pdf1 = m^-a1, pdf2 = m_br^(a2-a1) m^-a2
    I1 = (m_lo ** (1 - a1) - m_br ** (1 - a1)) / (a1 - 1)
    k2 = m_br ** (a2 - a1)
    I2 = k2 * (m_br ** (1 - a2) - m_hi ** (1 - a2)) / (a2 - 1)
    f1 = I1 / (I1 + I2)
    u = substream(seed, stream).random(n)
    m = np.empty(n)
    lo = u < f1
    # segment 1: invert  (m_lo^(1-a1) - m^(1-a1)) / (a1-1) = u (I1+I2)
    t = u[lo] * (I1 + I2)
    m[lo] = (m_lo ** (1 - a1) - t * (a1 - 1)) ** (1.0 / (1 - a1))
    t = (u[~lo] - f1) * (I1 + I2) / k2
    m[~lo] = (m_br ** (1 - a2) - t * (a2 - 1)) ** (1.0 / (1 - a2))
    return m


def merge_binaries(m_sun: np.ndarray, frac: float, seed: int):
    """5 % primordial binaries as centre-of-mass bodies (BASELINE.json configs 3-4):
    floor(frac N) seeded-random bodies get the sum of two IMF draws.  The log-uniform semi-major
    axis in [1e-5, 1e-2] is drawn (keeps the streams stable) and returned only for the record --
    nothing on the hot path sees it."""
    n = m_sun.size
    nb = int(np.floor(frac * n))
    rng = substream(seed, "binary")
    which = rng.choice(n, size=nb, replace=False)
    companion = kroupa_masses(nb, seed, stream="binary")  # second IMF draw, its own stream
    semi = 10.0 ** rng.uniform(-5.0, -2.0, size=nb)
    m = m_sun.copy()
    m[which] += companion
    return m, which, semi


# --------------------------------------------------------------------------- King (1966)

def _king_rho(W):
    W = np.maximum(W, 0.0)
    s = np.sqrt(W)
    return np.exp(W) * erf(s) - np.sqrt(4.0 * W / np.pi) * (1.0 + 2.0 * W / 3.0)


class KingModel:
    """King (1966) model of central dimensionless potential W0, tabulated and scaled to N-body
    units (G = M = 1, E = -1/4 via the model's own analytic potential energy; virial).

    Model units: r in King radii r0, velocities in sigma, 4 pi G rho0 = 9:
        W'' + (2/r) W' = -9 rho(W)/rho(W0),  W(0) = W0, W'(0) = 0,  G M(r) = -r^2 W'(r).
    """

    def __init__(self, W0: float = 9.0, ngrid: int = 8192):
        self.W0 = W0
        rho0 = _king_rho(W0)

        def rhs(r, y):
            return [y[1], -9.0 * _king_rho(y[0]) / rho0 - 2.0 * y[1] / r]

        def hit(r, y):
            return y[0]
        hit.terminal = True
        hit.direction = -1
        r_start = 1e-6
        y0 = [W0 - 1.5 * r_start ** 2, -3.0 * r_start]
        sol = solve_ivp(rhs, [r_start, 1e5], y0, events=hit, dense_output=True,
                        rtol=1e-11, atol=1e-13, method="DOP853")
        self.rt_model = float(sol.t_events[0][0])
        r = np.concatenate([[0.0], np.geomspace(1e-5, self.rt_model, ngrid - 1)])
        W = np.empty_like(r)
        dW = np.empty_like(r)
        W[0], dW[0] = W0, 0.0
        yy = sol.sol(np.maximum(r[1:], r_start))
        W[1:], dW[1:] = yy[0], yy[1]
        W[-1] = 0.0
        W = np.maximum(W, 0.0)
        Mr = -r * r * dW                       # G M(r), model units
        Mr = np.maximum.accumulate(Mr)
        rho_hat = _king_rho(W) / rho0          # rho / rho0
        dMdr = 9.0 * r * r * rho_hat           # 4 pi r^2 rho with 4 pi G rho0 = 9
        integrand = np.zeros_like(r)
        integrand[1:] = Mr[1:] / r[1:] * dMdr[1:]
        Wpot = -np.trapezoid(integrand, r)
        Mt = Mr[-1]
        # scale to G = M = 1, W_pot = -1/2
        self.len_scale = -2.0 * Wpot / (Mt * Mt)      # x_nb = x_model * len_scale
        self.vel_scale = np.sqrt(1.0 / (Mt * self.len_scale))
        self.r = r * self.len_scale
        self.W = W
        self.Mfrac = Mr / Mt
        # mass density in N-body units (total mass 1)
        rho = np.empty_like(r)
        rho[1:] = dMdr[1:] / (4.0 * np.pi * r[1:] ** 2) / Mt / self.len_scale ** 3
        rho[0] = 9.0 / (4.0 * np.pi) / Mt / self.len_scale ** 3      # rho_hat(0) = 1
        self.rho = rho
        self.r_core = self.len_scale          # King radius r0 in N-body units
        self.r_tidal = self.rt_model * self.len_scale

    def W_of_r(self, r):
        return np.interp(r, self.r, self.W)

    def mass_within(self, r):
        return np.interp(r, self.r, self.Mfrac)

    def density(self, r):
        return np.interp(r, self.r, self.rho)

    def smooth_field(self, x, v):
        """a0 = -M(<r) x / r^3 and its convective derivative along v (inputs only)."""
        r = np.sqrt(np.einsum("ij,ij->i", x, x))
        r = np.maximum(r, 1e-12)
        Mr = self.mass_within(r)
        g = Mr / r ** 3
        dg = 4.0 * np.pi * self.density(r) / r - 3.0 * Mr / r ** 4
        xv = np.einsum("ij,ij->i", x, v)
        a0 = -g[:, None] * x
        j0 = -(g[:, None] * v + (xv / r * dg)[:, None] * x)
        return a0, j0


def king_sample(n: int, model: KingModel, seed: int):
    """Positions by inverse M(r); speeds by rejection from p(v) ~ v^2 (exp(W - v^2/2) - 1),
    v < sqrt(2W) (sigma units), isotropic; scaled to N-body units."""
    u = substream(seed, "pos").random(n)
    u = np.clip(u, 1e-12, 1.0 - 1e-12)
    r = np.interp(u, model.Mfrac, model.r)
    x = r[:, None] * _isotropic(substream(seed, "dir"), n)
    W = np.maximum(model.W_of_r(r), 1e-12)
    rng = substream(seed, "vel")
    q = np.zeros(n)
    bound = np.where(W > 1.0, np.exp(W - 1.0) / np.maximum(W, 1.0), np.expm1(W))
    pending = np.arange(n)
    while pending.size:
        q1 = rng.random(pending.size)
        y = rng.random(pending.size) * bound[pending]
        Wp = W[pending]
        ok = y < q1 * q1 * np.expm1(Wp * (1.0 - q1 * q1))
        q[pending[ok]] = q1[ok]
        pending = pending[~ok]
    speed = q * np.sqrt(2.0 * W) * model.vel_scale
    v = speed[:, None] * _isotropic(substream(seed, "vdir"), n)
    return x, v


# --------------------------------------------------------------------------- block steps

def block_levels_uniform(n: int, kmin: int, kmax: int, seed: int) -> np.ndarray:
    return substream(seed, "level").integers(kmin, kmax + 1, size=n).astype(np.int32)


def block_levels_powerlaw(radius: np.ndarray, kmin: int, kmax: int, seed: int) -> np.ndarray:
    """Hermite-like occupancy: population of level k ~ 2^-(k-kmin); the deepest levels go to the
    innermost particles (deep blocks hold few particles), then a seeded +-1 level jitter."""
    n = radius.size
    ks = np.arange(kmin, kmax + 1)
    w = 2.0 ** (-(ks - kmin).astype(float))
    counts = np.floor(n * w / w.sum()).astype(np.int64)
    counts[0] += n - counts.sum()
    order = np.argsort(radius, kind="stable")          # innermost first
    lev_sorted = np.repeat(ks[::-1], counts[::-1])     # deepest level first
    lev = np.empty(n, dtype=np.int32)
    lev[order] = lev_sorted
    u = substream(seed, "jitter").random(n)
    lev = lev + (u < 0.25).astype(np.int32) - (u > 0.75).astype(np.int32)
    return np.clip(lev, kmin, kmax).astype(np.int32)


def t0_from_levels(levels: np.ndarray, t: float = 1.0) -> np.ndarray:
    """t0_j = t - 2^-k_j: the longest extrapolation each particle can see when every level is due."""
    return t - np.ldexp(1.0, -levels.astype(np.int64))


# --------------------------------------------------------------------------- neighbour radii

def h2_from_density(number_density: np.ndarray, n_target: float) -> np.ndarray:
    h = (3.0 * n_target / (4.0 * np.pi * number_density)) ** (1.0 / 3.0)
    return h * h


def knn_radius2(x: np.ndarray, k: int, factor: float = 1.01) -> np.ndarray:
    """(factor * distance to the k-th nearest other particle)^2 -- a geometric utility (KD-tree),
    used for config 1's h^2 at positions the caller supplies."""
    d, _ = cKDTree(x).query(x, k=k + 1)
    return (factor * d[:, k]) ** 2
