"""oracle.hermite_ac -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain numpy FP64 statement of the two-level Ahmad-Cohen (AC) neighbour scheme on top of the fourth-order
Hermite block-step integrator of oracle/hermite.py (readings R33-R38).
Forces come from the C oracle (oracle.regular / oracle.irregular).  Shares nothing with the CUDA path.

What the paper fixes:
  * P:49  "the AC neighbor scheme ... The full force of one particle is separated into two parts: regular
          and irregular forces.  The regular force is the summation of the forces from particles outside
          the neighbor radius and the irregular force accumulates only the neighbor forces.  Correspondingly
          there are regular (large) time steps and irregular (small) time steps ... During the irregular
          step, the regular force and its first order derivative calculated at the last regular step are
          used for the particle position and velocity prediction."
  * P:45  fourth-order Hermite, Aarseth step criterion;  P:47 block steps (powers of 0.5).
  * P:215 / Table A1: separate accuracy parameters eta_I (irregular) and eta_R (regular).
It prints no formula.  The scheme below is the textbook Hermite AC scheme (Makino & Aarseth 1992) with every
fill-in listed:

  R33  state of a body: x0, v0 at t0 (its last irregular time); irregular force aI, jI at t0 over its list L;
       regular force aR, jR at tR <= t0 (its last regular time); steps dtI <= dtR.  The predictor state handed
       to everybody else is the TOTAL  a0 = aI + aR + jR (t0 - tR),  j0 = jI + jR  (reading R2).
  R34  irregular step at t = t0 + dtI: aI1, jI1 = neighbour sums at the predicted state; the regular force is
       EXTRAPOLATED, aR(t) = aR + jR (t - tR), its derivative kept; Hermite corrector over dtI with the
       totals (the regular part being linear in t, its contribution to a2, a3 cancels exactly: the high-order
       terms are the irregular force's); new dtI from Aarseth's criterion on (aI1, jI1, a2, a3) with eta_I,
       block rule, never above dtR.
  R35  regular step at t = tR + dtR (always an irregular time of the body too): irregular force over the OLD
       list, total force with the NEW list (regular + irregular over L'), regular force w.r.t. the old list =
       total - irregular(old); irregular corrector as in R34 with the old list; REGULAR CORRECTION
       a2R, a3R = Hermite derivatives of the regular force over dtR,  x += a2R dtR^4/24 + a3R dtR^5/120,
       v += a2R dtR^3/6 + a3R dtR^4/24  (the terms the linear extrapolation left out); both force polynomials
       restart from the new list; new dtR from (aR_new, jR_new, a2R + dtR a3R, a3R) with eta_R, new dtI from the
       new-list irregular force with the irregular corrector's a2, a3.
  R36  a body with an EMPTY list has no irregular time scale: dtI = dtR (every step is a regular step).
  R37  start-up: dtR = initial_step(aR, jR), dtI = min(initial_step(aI, jI), dtR) (R36 if the list is empty).
  R38  neighbour radii are the caller's (no radius control, out of scope); a list that overflows its capacity
       would break regular + irregular = total, so overflow is an ERROR of the AC step (the caller shrinks h).

Pins (tests/test_hermite_ac_oracle.py): with every h2 = 0 the scheme IS the single-level integrator of
oracle/hermite.py (same states to rounding, same steps, same blocks); with every body a neighbour of every
other likewise; energy conservation with real radii, better with smaller eta; block invariants (dtI <= dtR,
regular times are irregular times, t0 a multiple of dtI, tR of dtR); a0 = aI + aR + jR (t0 - tR) at all
times; for a body whose list did not change at a regular step the old-list and new-list regular forces agree.
"""
from __future__ import annotations

import numpy as np

from . import hermite as H


def _forces(orc, m, st, t, idx, h2, cap, want_regular):
    """Irregular force over the CURRENT lists of bodies idx at time t; for want_regular also the regular
    force with radii h2 (new lists) and the irregular force over those new lists."""
    irr_old = orc.irregular(m, st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], t, idx, st["nnb"][idx],
                            st["list"][idx], cap)
    if not want_regular:
        return irr_old, None, None
    xp, vp = orc.predict(st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], t)
    reg = orc.regular(m, xp, vp, idx, h2[idx], cap)
    if reg["overflow"].any():
        raise OverflowError("neighbour list overflow during an AC step (reading R38)")
    irr_new = orc.irregular(m, st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], t, idx, reg["nnb"], reg["nblist"], cap)
    return irr_old, reg, irr_new


def _hermite_derivs(f0, d0, f1, d1, h):
    h = np.asarray(h, dtype=np.float64)[:, None]
    a2 = (-6.0 * (f0 - f1) - h * (4.0 * d0 + 2.0 * d1)) / h**2
    a3 = (12.0 * (f0 - f1) + 6.0 * h * (d0 + d1)) / h**3
    return a2, a3


def start(orc, m, x, v, h2, cap, eta_s, dt_max):
    """State at t = 0 (R33, R37)."""
    N = m.shape[0]
    idx = np.arange(N, dtype=np.int32)
    reg = orc.regular(m, x, v, idx, h2, cap)
    if reg["overflow"].any():
        raise OverflowError("neighbour list overflow at start-up (reading R38)")
    z3, z1 = np.zeros((N, 3)), np.zeros(N)
    irr = orc.irregular(m, x, v, z3, z3, z1, 0.0, idx, reg["nnb"], reg["nblist"], cap)
    dtR = H.initial_step(reg["acc"], reg["jerk"], eta_s, dt_max)
    dtI = np.minimum(H.initial_step(irr["acc"], irr["jerk"], eta_s, dt_max), dtR)
    dtI = np.where(reg["nnb"] == 0, dtR, dtI)
    return dict(x0=x.copy(), v0=v.copy(), t0=z1.copy(), aI=irr["acc"], jI=irr["jerk"], aR=reg["acc"], jR=reg["jerk"],
                tR=z1.copy(), dtI=dtI, dtR=dtR, a0=irr["acc"] + reg["acc"], j0=irr["jerk"] + reg["jerk"],
                nnb=reg["nnb"].copy(), list=reg["nblist"].copy())


def block_step(orc, m, st, h2, cap, eta_I, eta_R, dt_max, t_stop=np.inf):
    """One block of the two-level scheme, in place.  Returns (t, irregular-active indices, regular-active
    indices), or (t, None, None) with the state untouched if t > t_stop."""
    t, act = H.next_block(st["t0"], st["dtI"])
    if t > t_stop:
        return t, None, None
    due = st["tR"][act] + st["dtR"][act] == t
    reg_idx, irr_idx = act[due], act[~due]

    def irregular_corrector(idx, aI1, jI1):
        """R34: corrector over dtI with the extrapolated regular force; returns x1, v1, a2, a3, a1, j1."""
        aR_t = st["aR"][idx] + st["jR"][idx] * (t - st["tR"][idx])[:, None]
        a1, j1 = aI1 + aR_t, jI1 + st["jR"][idx]
        x1, v1, a2, a3 = H.correct(st["x0"][idx], st["v0"][idx], st["a0"][idx], st["j0"][idx], st["dtI"][idx], a1, j1)
        return x1, v1, a2, a3, a1, j1

    new = {}
    if irr_idx.size:
        io, _, _ = _forces(orc, m, st, t, irr_idx, h2, cap, False)
        x1, v1, a2, a3, a1, j1 = irregular_corrector(irr_idx, io["acc"], io["jerk"])
        dtR = st["dtR"][irr_idx]
        dtI = H.quantize_step(H.aarseth_step(io["acc"], io["jerk"], a2, a3, st["dtI"][irr_idx], eta_I), st["dtI"][irr_idx], t, dt_max)
        dtI = np.minimum(dtI, dtR)
        dtI = np.where(st["nnb"][irr_idx] == 0, dtR, dtI)
        new["irr"] = dict(x0=x1, v0=v1, aI=io["acc"], jI=io["jerk"], a0=a1, j0=j1, dtI=dtI)
    if reg_idx.size:
        io, rg, inw = _forces(orc, m, st, t, reg_idx, h2, cap, True)
        x1, v1, a2, a3, _, _ = irregular_corrector(reg_idx, io["acc"], io["jerk"])
        a_tot, j_tot = rg["acc"] + inw["acc"], rg["jerk"] + inw["jerk"]
        aR1_old, jR1_old = a_tot - io["acc"], j_tot - io["jerk"]                 # regular force w.r.t. the OLD list (R35)
        hR = st["dtR"][reg_idx]
        a2R, a3R = _hermite_derivs(st["aR"][reg_idx], st["jR"][reg_idx], aR1_old, jR1_old, hR)
        h = hR[:, None]
        x1 = x1 + (a2R * h**4 / 24.0 + a3R * h**5 / 120.0)
        v1 = v1 + (a2R * h**3 / 6.0 + a3R * h**4 / 24.0)
        dtR = H.quantize_step(H.aarseth_step(rg["acc"], rg["jerk"], a2R, a3R, hR, eta_R), hR, t, dt_max)
        dtI = H.quantize_step(H.aarseth_step(inw["acc"], inw["jerk"], a2, a3, st["dtI"][reg_idx], eta_I), st["dtI"][reg_idx], t, dt_max)
        dtI = np.minimum(dtI, dtR)
        dtI = np.where(rg["nnb"] == 0, dtR, dtI)
        new["reg"] = dict(x0=x1, v0=v1, aI=inw["acc"], jI=inw["jerk"], aR=rg["acc"], jR=rg["jerk"], a0=a_tot, j0=j_tot,
                          dtI=dtI, dtR=dtR, nnb=rg["nnb"], list=rg["nblist"], aR1_old=aR1_old)
    # every active body is advanced at once, from forces evaluated at the pre-step state of everybody
    if irr_idx.size:
        for k, v in new["irr"].items():
            st[k][irr_idx] = v
        st["t0"][irr_idx] = t
    if reg_idx.size:
        for k, v in new["reg"].items():
            if k != "aR1_old":
                st[k][reg_idx] = v
        st["t0"][reg_idx] = t
        st["tR"][reg_idx] = t
        st["_last_reg"] = (reg_idx, new["reg"]["aR1_old"])
    return t, act, reg_idx


def integrate(orc, m, x, v, h2, cap, t_end, eta_I, eta_R, eta_s, dt_max, on_block=None):
    """Two-level AC integration from t = 0 to t_end (a multiple of dt_max).  Returns the state and counters."""
    st = start(orc, m, x, v, h2, cap, eta_s, dt_max)
    blocks = isteps = rsteps = 0
    while True:
        t, act, reg = block_step(orc, m, st, h2, cap, eta_I, eta_R, dt_max, t_stop=t_end)
        if act is None:
            break
        blocks += 1
        isteps += act.size
        rsteps += reg.size
        if on_block is not None:
            on_block(t, act, reg, st)
    st.update(blocks=blocks, irregular_steps=isteps, regular_steps=rsteps)
    return st
