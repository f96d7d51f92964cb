"""oracle.hermite -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy FP64 statement of the steps either side of the regular-force pass:
block selection, the fourth-order Hermite corrector, the new block time step, and a small
block-step integrator built from them.  Shares nothing with ``paper_1504_03687_b200``.

What the paper fixes and what it leaves open (readings R27-R31):
  * P:45  "NBODY6 uses the fourth-order Hermite integration method" (Makino 1991) -- the paper prints
          no formula; the corrector below is the textbook one it names: the acceleration over a step
          is the cubic Hermite interpolant of (a0, j0) at t0 and (a1, j1) at t1 = t0 + dt, and the
          corrector adds that cubic's second- and third-derivative terms to the predicted x, v.
  * P:47  "particle time steps are adjusted to quantized values, usually an integer power of 0.5 ...
          at each time step, active particles (the particles that satisfy the time step criterion)
          are integrated together" -- block steps: dt = 2^-k, t0 a multiple of dt.
  * P:89  section 3.3.1: active particles are selected from an index list sorted by time step with boundary
          offsets I_off(i); ``next_block`` is the definition that algorithm implements
          (active <=> t0 + dt = min_j (t0_j + dt_j)); ``sorted_list_prefix`` is the paper's list.
  * time step criterion: the paper only names "the standard Aarseth scheme" and eta;
          the criterion below is Aarseth's (1985) as used with the Hermite scheme (Makino & Aarseth 1992).

Pins (tests/test_hermite_oracle.py): a motion whose acceleration is exactly a cubic polynomial in t
is reproduced exactly (rational arithmetic); a2, a3 are that polynomial's derivatives; a circular
Kepler orbit with a shared step shows fourth-order convergence of the energy error; the active set
equals the prefix of the paper's step-sorted list; block-step invariants (t0 multiple of dt, steps at
most double, doubling only at commensurate times) hold along an integration; a Plummer sphere
conserves energy.  ``aarseth_step``: for harmonic motion a(t) = A cos(wt) e the criterion is exactly
sqrt(eta) / w at every phase and amplitude (closed form), plus two cases worked by hand with a2 handed
in at the start of the step (so "a2 advanced by dt a3" is pinned); ``initial_step``: hand cases on and
off a power of two and at the dt_max cap; the degenerate-criterion rule R32 (dt_req = 0 / NaN keeps
the step, nothing falls below dt_max 2^-40) on hand cases.  tests/test_oracle_mutations.py applies 22 single-term
mutations to correct / aarseth_step / quantize_step / initial_step (no sqrt, swapped or dropped products, wrong powers,
a2 at the start, ceil for floor, ...) and checks that each makes a pin fail.
"""
from __future__ import annotations

import numpy as np


# ----------------------------------------------------------------------------- block selection

def next_block(t0: np.ndarray, dt: np.ndarray):
    """t_next = min_j (t0_j + dt_j); active = {j : t0_j + dt_j == t_next}, ascending.  Exact: block
    times are dyadic rationals, t0 + dt is computed without rounding."""
    tn = t0 + dt
    t_next = tn.min()
    return float(t_next), np.flatnonzero(tn == t_next).astype(np.int32)


def sorted_list_prefix(dt: np.ndarray, t_next: float):
    """The paper's sorting-list statement (Figures 1-2): indices sorted by step, smallest first;
    the active particles at block time t_next are the prefix holding every step 0.5^i that divides
    t_next.  Returns that prefix as a sorted index array (valid when every t0 is a multiple of dt)."""
    order = np.argsort(dt, kind="stable")
    divides = np.array([(t_next / d) == np.floor(t_next / d) for d in dt[order]])
    # steps ascend along the list, so "divides" is a run of True followed by False
    n = int(divides.sum())
    assert divides[:n].all() and not divides[n:].any()
    return np.sort(order[:n]).astype(np.int32)


# ----------------------------------------------------------------------------- corrector

def correct(x0, v0, a0, j0, dt, a1, j1):
    """Fourth-order Hermite corrector.  Inputs [n][3] (dt [n]): state, acceleration and jerk at t0,
    acceleration and jerk at t1 = t0 + dt (evaluated at the predicted x, v).  Returns
    x1, v1 (corrected), a2 (second derivative of the acceleration at t0), a3 (third, constant)."""
    h = np.asarray(dt, dtype=np.float64)[:, None]
    a2 = (-6.0 * (a0 - a1) - h * (4.0 * j0 + 2.0 * j1)) / h**2
    a3 = (12.0 * (a0 - a1) + 6.0 * h * (j0 + j1)) / h**3
    x1 = x0 + v0 * h + a0 * h**2 / 2.0 + j0 * h**3 / 6.0 + a2 * h**4 / 24.0 + a3 * h**5 / 120.0
    v1 = v0 + a0 * h + j0 * h**2 / 2.0 + a2 * h**3 / 6.0 + a3 * h**4 / 24.0
    return x1, v1, a2, a3


# ----------------------------------------------------------------------------- time step

def _norm(a):
    return np.sqrt((a * a).sum(axis=1))


def aarseth_step(a1, j1, a2_0, a3, dt, eta):
    """Aarseth's criterion with the derivatives at the END of the step (a2 advanced by dt a3):
    dt_req = sqrt( eta (|a||a2| + |j|^2) / (|j||a3| + |a2|^2) )."""
    a2 = a2_0 + np.asarray(dt)[:, None] * a3
    na, nj, n2, n3 = _norm(a1), _norm(j1), _norm(a2), _norm(a3)
    with np.errstate(divide="ignore", invalid="ignore"):        # 0/0 (no force at all) -> NaN: handled by quantize_step (R32)
        return np.sqrt(eta * (na * n2 + nj * nj) / (nj * n3 + n2 * n2))


DT_MIN_LEVELS = 40      # reading R32: no step below dt_max * 2^-40


def quantize_step(dt_req, dt_old, t1, dt_max, dt_min=None):
    """Block-step rule (steps are integer powers of 0.5).  Candidate = dt_old; it is doubled once
    if dt_req >= 2 dt_old, 2 dt_old <= dt_max and t1 is a multiple of 2 dt_old (so that t0 stays a
    multiple of dt); otherwise it is halved while it exceeds dt_req.
    Degenerate criterion (reading R32; the paper is silent): dt_req = 0 or NaN (a body with
    a1 = j1 = 0, or every derivative zero) carries no information -- the step is KEPT; and no step is
    halved below dt_min = dt_max 2^-40, so the block loop can never stall on a vanishing step."""
    dt_req = np.asarray(dt_req, dtype=np.float64)
    out = np.array(dt_old, dtype=np.float64, copy=True)
    if dt_min is None:
        dt_min = dt_max * 2.0 ** -DT_MIN_LEVELS
    for k in range(out.shape[0]):
        d = out[k]
        if not dt_req[k] > 0.0:                 # 0 or NaN: keep the step
            continue
        if dt_req[k] >= 2.0 * d and 2.0 * d <= dt_max and (t1 / (2.0 * d)) == np.floor(t1 / (2.0 * d)):
            d = 2.0 * d
        else:
            while d > dt_req[k] and d > dt_min:
                d *= 0.5
        out[k] = d
    return out


def initial_step(a, j, eta_s, dt_max):
    """Start-up step: the largest power of 0.5 not above min(eta_s |a| / |j|, dt_max), and not below
    dt_max 2^-40; |a| = |j| = 0 (no information: NaN) gives dt_max (reading R32)."""
    with np.errstate(divide="ignore", invalid="ignore"):
        req = eta_s * _norm(a) / _norm(j)
    req = np.where(np.isnan(req), dt_max, req)
    req = np.clip(req, dt_max * 2.0 ** -DT_MIN_LEVELS, dt_max)
    return 2.0 ** np.floor(np.log2(req))


# ----------------------------------------------------------------------------- a small block-step integrator

def integrate(m, x, v, t_end, eta, eta_s, dt_max, force):
    """Hermite block-step integration from t = 0 to t_end (a multiple of dt_max) with the TOTAL force.
    ``force(m, xp, vp, idx) -> (acc[n][3], jerk[n][3])`` evaluates the active block at the predicted
    state of all bodies (the oracle's direct sum with h2 = 0 in the tests).  Returns the final state
    dict and counters."""
    N = m.shape[0]
    x0, v0 = x.copy(), v.copy()
    a0, j0 = force(m, x0, v0, np.arange(N, dtype=np.int32))
    t0 = np.zeros(N)
    dt = initial_step(a0, j0, eta_s, dt_max)
    blocks = psteps = 0
    while True:
        t, idx = next_block(t0, dt)
        if t > t_end:
            break
        h = (t - t0)[:, None]
        xp = x0 + v0 * h + a0 * h**2 / 2.0 + j0 * h**3 / 6.0          # predictor, reading R2
        vp = v0 + a0 * h + j0 * h**2 / 2.0
        a1, j1 = force(m, xp, vp, idx)
        x1, v1, a2, a3 = correct(x0[idx], v0[idx], a0[idx], j0[idx], dt[idx], a1, j1)
        req = aarseth_step(a1, j1, a2, a3, dt[idx], eta)
        dt[idx] = quantize_step(req, dt[idx], t, dt_max)
        x0[idx], v0[idx], a0[idx], j0[idx], t0[idx] = x1, v1, a1, j1, t
        blocks += 1
        psteps += idx.shape[0]
    return dict(x0=x0, v0=v0, a0=a0, j0=j0, t0=t0, dt=dt, blocks=blocks, particle_steps=psteps)
