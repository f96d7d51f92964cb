"""SURVEY 8(f) NEXT-3 on the GPU (block selection, Hermite corrector, block time step) against
oracle/hermite.py, element by element on the same seeded inputs, and a closed block loop
(select -> predict -> regular force -> correct) checked for energy conservation and against the
oracle's own integration.  Needs a B200."""
import numpy as np
import pytest

import nbgen
from oracle import hermite as H

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def _open(cfg, cap=8):
    import paper_1504_03687_b200 as nb
    ctx = nb.nb_open(cfg["N"], cap)
    nb.nb_set_j(ctx, *(_dev(cfg[k]) for k in ("m", "x0", "v0", "a0", "j0", "t0")))
    return ctx


def _state(ctx, with_steps=True):
    ctx_state = ctx.get_state(with_steps)
    ctx.synchronize()
    return {k: v.cpu().numpy() for k, v in ctx_state.items()}


def test_next_block_matches_the_definition_and_is_ascending():
    cfg = nbgen.make_config(2, N=70001, n_i=16)
    ctx = _open(cfg)
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    ctx.set_steps(_dev(dt))
    idx = torch.empty(cfg["N"], dtype=torch.int32, device="cuda")
    t_next, n = ctx.next_block(idx)
    t_ref, act = H.next_block(cfg["t0"], dt)
    assert t_next == t_ref and n == act.size
    assert np.array_equal(idx[:n].cpu().numpy(), act)                  # ascending, like the oracle's
    # a second time level: only the deepest level is due
    t0 = np.floor(0.3 / dt) * dt
    cfg2 = dict(cfg, t0=t0)
    ctx2 = _open(cfg2)
    ctx2.set_steps(_dev(dt))
    t_next, n = ctx2.next_block(idx)
    t_ref, act = H.next_block(t0, dt)
    assert t_next == t_ref and n == act.size and np.array_equal(idx[:n].cpu().numpy(), act)
    assert np.array_equal(act, H.sorted_list_prefix(dt, t_ref))        # = the paper's step-sorted prefix
    ctx.close(); ctx2.close()


def test_init_steps_match_the_oracle():
    cfg = nbgen.make_config(2, N=20000, n_i=16)
    ctx = _open(cfg)
    ctx.init_steps(0.02, 2.0**-3)
    got = _state(ctx)["dt"]
    ref = H.initial_step(cfg["a0"], cfg["j0"], 0.02, 2.0**-3)
    assert np.array_equal(got, ref)
    ctx.close()


def test_corrector_and_new_step_match_the_oracle():
    rng = np.random.default_rng(11)
    cfg = nbgen.make_config(2, N=30000, n_i=16)
    N = cfg["N"]
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    cfg = dict(cfg, t0=np.floor(0.3 / dt) * dt)             # mid-run: only the deepest level is due next
    ctx = _open(cfg)
    ctx.set_steps(_dev(dt))
    t, act = H.next_block(cfg["t0"], dt)
    n = act.size
    assert 1000 < n < N // 2
    # new forces of the right magnitude: the old ones advanced by the jerk plus a perturbation, so that
    # all three branches of the step rule (double / keep / halve) occur
    a1 = cfg["a0"][act] + cfg["j0"][act] * dt[act, None] * (1 + 0.3 * rng.standard_normal((n, 3)))
    j1 = cfg["j0"][act] * (1 + rng.standard_normal((n, 3)) * rng.choice([0.01, 0.3, 3.0], size=(n, 1)))
    eta, dt_max = 0.02, 2.0**-6
    ctx.correct(t, _dev(act), _dev(a1), _dev(j1), eta, dt_max)
    got = _state(ctx)
    x1, v1, a2, a3 = H.correct(cfg["x0"][act], cfg["v0"][act], cfg["a0"][act], cfg["j0"][act], dt[act], a1, j1)
    req = H.aarseth_step(a1, j1, a2, a3, dt[act], eta)
    new = H.quantize_step(req, dt[act], t, dt_max)
    assert np.abs(got["x0"][act] - x1).max() <= 1e-14 * np.abs(x1).max()
    assert np.abs(got["v0"][act] - v1).max() <= 1e-14 * np.abs(v1).max()
    assert np.array_equal(got["a0"][act], a1) and np.array_equal(got["j0"][act], j1)
    assert np.all(got["t0"][act] == t)
    # the step is a floating-point decision taken in FP64 on both sides: identical except where dt_req
    # sits within rounding of a power of two (none expected)
    edge = np.abs(req / 2.0 ** np.round(np.log2(req)) - 1.0) < 1e-12
    assert np.array_equal(got["dt"][act][~edge], new[~edge]) and edge.sum() <= 1
    kinds = np.sign(np.log2(new / dt[act]))
    assert (kinds > 0).any() and (kinds == 0).any() and (kinds < 0).any()
    # everybody else untouched
    rest = np.setdiff1d(np.arange(N), act)
    for k in ("x0", "v0", "a0", "j0", "t0"):
        assert np.array_equal(got[k][rest], cfg[k][rest])
    assert np.array_equal(got["dt"][rest], dt[rest])
    ctx.close()


def _oracle_force(m, xp, vp, idx):
    import oracle
    out = oracle.regular(m, xp, vp, idx, np.zeros(idx.shape[0]), 8)
    return out["acc"], out["jerk"]


def test_block_loop_conserves_energy_and_follows_the_oracle_integration():
    """N = 1024 Plummer sphere from t = 0 to 1/8 with the total force (nb_regular, h2 = 0): the GPU loop
    next_block -> predict_all -> regular -> correct against oracle.hermite.integrate with the FP64 direct sum."""
    import paper_1504_03687_b200 as nb
    N, cap = 1024, 8
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    eta, eta_s, dt_max, t_end = 0.01, 0.01, 2.0**-4, 0.125
    ref = H.integrate(m, x, v, t_end, eta, eta_s, dt_max, _oracle_force)

    ctx = nb.nb_open(N, cap)
    kw = dict(dtype=torch.float64, device="cuda")
    buf = dict(acc=torch.empty((N, 3), **kw), jerk=torch.empty((N, 3), **kw), pot=torch.empty(N, **kw),
               nnb=torch.empty(N, dtype=torch.int32, device="cuda"),
               nblist=torch.empty((N, cap), dtype=torch.int32, device="cuda"),
               overflow=torch.empty(N, dtype=torch.int32, device="cuda"))
    view = lambda n: {k: (b[:n] if b.dim() == 1 else b[:n]) for k, b in buf.items()}
    zeros_h2 = torch.zeros(N, **kw)
    all_idx = torch.arange(N, dtype=torch.int32, device="cuda")
    zero3 = torch.zeros((N, 3), **kw)

    def total_force_and_energy(t):
        ctx.predict_all(t)
        ctx.regular(all_idx, zeros_h2, **buf)
        ctx.synchronize()
        st = _state(ctx, with_steps=False)
        e = 0.5 * (st["m"] * (st["v0"] ** 2).sum(1)).sum() + 0.5 * (st["m"] * buf["pot"].cpu().numpy()).sum()
        return e

    # start-up: forces at t = 0 through the library itself, then the initial steps
    nb.nb_set_j(ctx, _dev(m), _dev(x), _dev(v), zero3, zero3, torch.zeros(N, **kw))
    e0 = total_force_and_energy(0.0)
    nb.nb_set_j(ctx, _dev(m), _dev(x), _dev(v), buf["acc"].clone(), buf["jerk"].clone(), torch.zeros(N, **kw))
    ctx.init_steps(eta_s, dt_max)
    idx = torch.empty(N, dtype=torch.int32, device="cuda")
    blocks = psteps = 0
    while True:
        t, n = ctx.next_block(idx)
        if t > t_end:
            break
        ctx.predict_all(t)
        o = view(n)
        ctx.regular(idx[:n], zeros_h2[:n], **o)
        ctx.correct(t, idx[:n], o["acc"], o["jerk"], eta, dt_max)
        blocks += 1
        psteps += n
    st = _state(ctx)
    assert np.all(st["t0"] == t_end)
    e1 = total_force_and_energy(t_end)
    print("block loop: blocks", blocks, "particle steps", psteps, "oracle", ref["blocks"], ref["particle_steps"],
          "dE/E", (e1 - e0) / e0, "max |dx|", np.abs(st["x0"] - ref["x0"]).max())
    assert abs((e1 - e0) / e0) < 5e-6
    # FP32 pair arithmetic perturbs the forces by ~1e-7; a step decision may flip now and then
    assert abs(psteps - ref["particle_steps"]) <= 0.01 * ref["particle_steps"]
    assert np.abs(st["x0"] - ref["x0"]).max() < 1e-5 and np.abs(st["v0"] - ref["v0"]).max() < 1e-4
    ctx.close()


def test_ac_split_block_loop_at_65536_bodies_follows_the_oracle():
    """Three consecutive blocks of a 65536-body cluster with the Ahmad-Cohen split evaluated at the block
    time: nb_regular (neighbours excluded, lists emitted) + nb_irregular (the listed neighbours, FP64)
    added by the caller = total force -> nb_correct.  The oracle runs the same three blocks with its own
    regular, irregular, corrector and step rule; states must agree."""
    import oracle
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(2)
    N, cap = cfg["N"], cfg["cap"]
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    st = dict(m=cfg["m"], x0=cfg["x0"].copy(), v0=cfg["v0"].copy(), a0=cfg["a0"].copy(), j0=cfg["j0"].copy(),
              t0=np.floor(0.3 / dt) * dt, dt=dt.copy())
    eta, dt_max = 0.02, 2.0**-6
    ctx = nb.nb_open(N, cap)
    nb.nb_set_j(ctx, *(_dev(st[k]) for k in ("m", "x0", "v0", "a0", "j0", "t0")))
    ctx.set_steps(_dev(st["dt"]))
    h2_np = np.minimum(cfg["h2_all"], 0.01)        # halo bodies would get radii that swallow the core: keep every row under cap
    h2_all = _dev(h2_np)
    idx = torch.empty(N, dtype=torch.int32, device="cuda")
    sizes = []
    for _ in range(3):
        # ---- GPU
        t, n = ctx.next_block(idx)
        act = idx[:n]
        ctx.predict_all(t)
        reg = ctx.regular_alloc(act, h2_all[act.long()].contiguous())
        irr = dict(acc=torch.empty_like(reg["acc"]), jerk=torch.empty_like(reg["jerk"]))
        ctx.irregular(t, act, reg["nnb"], reg["nblist"], **irr)
        ctx.correct(t, act, reg["acc"] + irr["acc"], reg["jerk"] + irr["jerk"], eta, dt_max)
        # ---- oracle
        t_ref, a_ref = H.next_block(st["t0"], st["dt"])
        assert t == t_ref and np.array_equal(act.cpu().numpy(), a_ref)
        xp, vp = oracle.predict(st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], t_ref)
        r = oracle.regular(st["m"], xp, vp, a_ref, h2_np[a_ref], cap)
        assert not r["overflow"].any() and np.array_equal(r["nnb"], reg["nnb"].cpu().numpy())
        i = oracle.irregular(st["m"], st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], t_ref, a_ref, r["nnb"],
                             r["nblist"], cap)
        assert np.abs(i["acc"] - r["acc_nb"]).max() <= 1e-12 * np.abs(i["acc"]).max()   # same sum, two routes
        a1, j1 = r["acc"] + i["acc"], r["jerk"] + i["jerk"]
        x1, v1, a2, a3 = H.correct(st["x0"][a_ref], st["v0"][a_ref], st["a0"][a_ref], st["j0"][a_ref],
                                   st["dt"][a_ref], a1, j1)
        new = H.quantize_step(H.aarseth_step(a1, j1, a2, a3, st["dt"][a_ref], eta), st["dt"][a_ref], t_ref, dt_max)
        st["x0"][a_ref], st["v0"][a_ref], st["a0"][a_ref], st["j0"][a_ref] = x1, v1, a1, j1
        st["t0"][a_ref], st["dt"][a_ref] = t_ref, new
        sizes.append(n)
    got = _state(ctx)
    assert len(set(sizes)) > 1 and max(sizes) > 1000 and min(sizes) >= 1      # a deep block and tiny follow-ups
    assert np.array_equal(got["t0"], st["t0"])
    assert np.abs(got["x0"] - st["x0"]).max() < 1e-12 and np.abs(got["v0"] - st["v0"]).max() < 1e-10
    assert np.abs(got["a0"] - st["a0"]).max() <= 1e-5 * np.abs(st["a0"]).max()
    flips = (got["dt"] != st["dt"]).sum()
    print("AC-split loop: block sizes", sizes, "step decisions that differ", int(flips))
    assert flips <= 1e-3 * sum(sizes)      # FP32 pair terms move dt_req by ~1e-7: a flip needs dt_req that close to 2^-k
    ctx.close()


# ----------------------------------------------------------------------------- nb_block_step (one call per block)

def _oracle_block(st, m, eta, dt_max, h2_np=None, cap=None):
    """One block step of the oracle on the state dict st (in place): selection, predictor, total force
    (regular with h2 = 0, or regular + irregular on the oracle's own lists), corrector, new step."""
    import oracle
    t, act = H.next_block(st["t0"], st["dt"])
    xp, vp = oracle.predict(st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], t)
    if h2_np is None:
        r = oracle.regular(m, xp, vp, act, np.zeros(act.size), 8, want_list=False)
        a1, j1, nnb = r["acc"], r["jerk"], None
    else:
        r = oracle.regular(m, xp, vp, act, h2_np[act], cap)
        i = oracle.irregular(m, st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], t, act, r["nnb"], r["nblist"], cap)
        a1, j1, nnb = r["acc"] + i["acc"], r["jerk"] + i["jerk"], r["nnb"]
    x1, v1, a2, a3 = H.correct(st["x0"][act], st["v0"][act], st["a0"][act], st["j0"][act], st["dt"][act], a1, j1)
    new = H.quantize_step(H.aarseth_step(a1, j1, a2, a3, st["dt"][act], eta), st["dt"][act], t, dt_max)
    st["x0"][act], st["v0"][act], st["a0"][act], st["j0"][act] = x1, v1, a1, j1
    st["t0"][act], st["dt"][act] = t, new
    return t, act, nnb


def test_block_step_200_blocks_at_65536_in_lockstep_with_the_oracle():
    """nb_block_step (selection -> fused prediction + regular force -> corrector, one call
    and one host read-back per block) for 200 consecutive blocks of a 65536-body cluster with power-law block
    occupancy (deep levels hold few bodies), against the oracle doing the same 200 blocks.  Active sets
    must be identical block by block; a step decision may flip where dt_req sits within FP32 force rounding
    of a power of two -- flips are counted and adopted so that the two runs stay comparable."""
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(3, N=65536)
    N = cfg["N"]
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    st = dict(x0=cfg["x0"].copy(), v0=cfg["v0"].copy(), a0=cfg["a0"].copy(), j0=cfg["j0"].copy(),
              t0=np.floor(0.3 / dt) * dt, dt=dt.copy())
    m = cfg["m"]
    eta, dt_max = 0.02, 2.0**-6
    ctx = nb.nb_open(N, 8)
    nb.nb_set_j(ctx, *(_dev(a) for a in (m, st["x0"], st["v0"], st["a0"], st["j0"], st["t0"])))
    ctx.set_steps(_dev(st["dt"]))
    sizes, flips, fused = [], 0, 0
    for b in range(200):
        t, n = ctx.block_step(None, eta, dt_max)
        fused += ctx.info("last_fused")
        t_ref, act, _ = _oracle_block(st, m, eta, dt_max)
        blk = ctx.get_block(n)
        assert t == t_ref and n == act.size, (b, t, t_ref, n, act.size)
        assert np.array_equal(blk["idx_act"].cpu().numpy(), act), b
        sizes.append(n)
        # adopt flipped step decisions so the runs stay in lockstep.  (a2 ~ (a0 - a1) / dt^2 amplifies the FP32
        # rounding of the force at tiny steps: dt_req moves by ~1e-3 relative, so a body whose dt_req sits that
        # close to a power of two may decide differently)
        g_dt = _state(ctx)["dt"]
        diff = np.flatnonzero(g_dt != st["dt"])
        assert np.isin(diff, act).all()
        flips += diff.size
        st["dt"][diff] = g_dt[diff]
    got = _state(ctx)
    print("block_step x200: sizes min/median/max", min(sizes), int(np.median(sizes)), max(sizes), "particle steps",
          sum(sizes), "flips", flips, "fused blocks", fused)
    assert min(sizes) < 128 and fused > 50                       # small deep blocks took the fused path
    assert flips <= max(2, int(1e-3 * sum(sizes)))
    assert np.array_equal(got["t0"], st["t0"])
    # the corrector turns a force error da into dx ~ 0.35 da dt^2 and dv ~ 1.5 da dt per step; the FP32 pair
    # arithmetic gives da <~ 1e-6 |a|, and the Kroupa cluster has bodies with |a| ~ 1e3 next to a heavy neighbour
    # on steps up to 2^-8: dx <~ 5e-9, dv <~ 6e-6 in the worst case
    ex, ev = np.abs(got["x0"] - st["x0"]).max(), np.abs(got["v0"] - st["v0"]).max()
    print("block_step x200: max |dx|", ex, "max |dv|", ev, "max |a|", np.abs(st["a0"]).max())
    assert ex < 5e-9 and ev < 6e-6
    scale = np.linalg.norm(st["a0"], axis=1)
    assert np.max(np.linalg.norm(got["a0"] - st["a0"], axis=1) / scale) <= 1e-5
    ctx.close()


def test_block_step_with_neighbour_radii_adds_the_irregular_force():
    """nb_block_step with h2_all: regular force with lists + neighbour force on those lists, added in place
    (P:49), then the corrector -- five blocks against the oracle's regular + irregular + corrector; the
    block's own buffers (nb_get_block) carry the total force and the neighbour counts."""
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(2, N=20000, n_i=16)
    N, cap = cfg["N"], cfg["cap"]
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    st = dict(x0=cfg["x0"].copy(), v0=cfg["v0"].copy(), a0=cfg["a0"].copy(), j0=cfg["j0"].copy(),
              t0=np.floor(0.3 / dt) * dt, dt=dt.copy())
    m = cfg["m"]
    h2_np = np.minimum(cfg["h2_all"], 0.01)
    eta, dt_max = 0.02, 2.0**-6
    ctx = nb.nb_open(N, cap)
    nb.nb_set_j(ctx, *(_dev(a) for a in (m, st["x0"], st["v0"], st["a0"], st["j0"], st["t0"])))
    ctx.set_steps(_dev(st["dt"]))
    h2_d = _dev(h2_np)
    for b in range(5):
        t, n = ctx.block_step(h2_d, eta, dt_max)
        before = {k: st[k].copy() for k in ("a0", "j0")}
        t_ref, act, nnb = _oracle_block(st, m, eta, dt_max, h2_np, cap)
        blk = ctx.get_block(n, want_list=True)
        assert t == t_ref and np.array_equal(blk["idx_act"].cpu().numpy(), act)
        assert np.array_equal(blk["nnb"].cpu().numpy(), nnb) and nnb.max() <= cap and nnb.max() > 0
        a1 = st["a0"][act]
        assert np.abs(blk["acc"].cpu().numpy() - a1).max() <= 1e-5 * np.abs(a1).max()
    got = _state(ctx)
    assert np.array_equal(got["t0"], st["t0"])
    assert np.abs(got["x0"] - st["x0"]).max() < 1e-11 and np.abs(got["v0"] - st["v0"]).max() < 1e-9
    assert (got["dt"] != st["dt"]).sum() <= 2
    ctx.close()


def test_block_step_stops_at_t_stop_and_closed_loop_conserves_energy():
    """The closed loop of test_block_loop_... driven by nb_block_step alone: N = 1024 Plummer sphere to
    t = 1/8; t_stop leaves the state untouched once nothing is due; energy conserved; same particle steps
    as the oracle integration."""
    import paper_1504_03687_b200 as nb
    N = 1024
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    eta, eta_s, dt_max, t_end = 0.01, 0.01, 2.0**-4, 0.125
    ref = H.integrate(m, x, v, t_end, eta, eta_s, dt_max, _oracle_force)
    ctx = nb.nb_open(N, 8)
    kw = dict(dtype=torch.float64, device="cuda")
    z3, z1 = torch.zeros((N, 3), **kw), torch.zeros(N, **kw)
    all_idx = torch.arange(N, dtype=torch.int32, device="cuda")

    def energy(t):
        ctx.predict_all(t)
        out = ctx.regular_alloc(all_idx, z1)
        ctx.synchronize()
        s_ = _state(ctx, with_steps=False)
        return 0.5 * (s_["m"] * (s_["v0"] ** 2).sum(1)).sum() + 0.5 * (s_["m"] * out["pot"].cpu().numpy()).sum(), out

    nb.nb_set_j(ctx, _dev(m), _dev(x), _dev(v), z3, z3, z1)
    e0, out = energy(0.0)
    nb.nb_set_j(ctx, _dev(m), _dev(x), _dev(v), out["acc"].clone(), out["jerk"].clone(), z1)
    ctx.init_steps(eta_s, dt_max)
    blocks = psteps = 0
    for _ in range(40):                                                   # one call per block ...
        t, n = ctx.block_step(None, eta, dt_max, t_stop=t_end)
        assert n > 0
        blocks += 1
        psteps += n
    t, b2, p2 = ctx.run_blocks(None, eta, dt_max, t_stop=t_end)           # ... and the loop inside the library
    assert t > t_end and b2 > 0
    blocks += b2; psteps += p2
    s1 = _state(ctx)
    t2, n2 = ctx.block_step(None, eta, dt_max, t_stop=t_end)            # again: still nothing due, state untouched
    s2 = _state(ctx)
    assert n2 == 0 and t2 == t and all(np.array_equal(s1[k], s2[k]) for k in s1)
    assert np.all(s1["t0"] == t_end)
    e1, _ = energy(t_end)
    print("block_step loop: blocks", blocks, "particle steps", psteps, "oracle", ref["blocks"], ref["particle_steps"],
          "dE/E", (e1 - e0) / e0)
    assert abs((e1 - e0) / e0) < 5e-6
    assert abs(psteps - ref["particle_steps"]) <= 0.01 * ref["particle_steps"]
    assert np.abs(s1["x0"] - ref["x0"]).max() < 1e-5
    ctx.close()


def test_selection_from_chunk_minima_equals_the_full_scan():
    """The block loops keep min (t0 + dt) per 2048-body chunk and rescan only the chunks the last corrector
    touched (section 3.3.1: the search for the due particles must not cost O(N) per block).  Same blocks,
    bit-identical state as with the full scan (NB_TUNE_SELECT_CHUNKS = 0) -- over single calls and batched
    loops, and after the state and the steps were replaced from outside the chain (nb_update_j with new t0,
    nb_set_steps), which must invalidate every stored minimum.  N spans several chunks and a ragged one."""
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(3, N=20000, n_i=16)
    N = cfg["N"]
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    t0 = np.floor(0.3 / dt) * dt
    eta, dt_max = 0.02, 2.0**-6
    rng = np.random.default_rng(5)
    upd = np.sort(rng.choice(N, 37, replace=False)).astype(np.int32)

    def run(chunks):
        ctx = nb.nb_open(N, 8)
        ctx.tune("select_chunks", chunks)
        nb.nb_set_j(ctx, *(_dev(a) for a in (cfg["m"], cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], t0)))
        ctx.set_steps(_dev(dt))
        log = []
        for _ in range(25):
            log.append(ctx.block_step(None, eta, dt_max))
        log.append(ctx.run_blocks(None, eta, dt_max, t_stop=1.0e9, max_blocks=40))
        # replace 37 bodies (earlier t0: they become the next block) and then every step
        s = _state(ctx)
        t_now = log[-1][0]
        ctx.update_j(_dev(upd), *(_dev(a) for a in (cfg["m"][upd], s["x0"][upd], s["v0"][upd], s["a0"][upd], s["j0"][upd],
                                                    np.full(upd.size, t_now - 2.0**-9))))
        log.append(ctx.block_step(None, eta, dt_max))
        log.append(ctx.run_blocks(None, eta, dt_max, t_stop=1.0e9, max_blocks=10))
        ctx.set_steps(_dev(np.minimum(_state(ctx)["dt"], 2.0**-12)))
        for _ in range(6):
            log.append(ctx.block_step(None, eta, dt_max))
        log.append(ctx.run_blocks(None, eta, dt_max, t_stop=1.0e9, max_blocks=30))
        out = _state(ctx)
        ctx.close()
        return log, out

    log1, s1 = run(1)
    log0, s0 = run(0)
    assert log1 == log0
    assert 0 < log1[26][1] <= upd.size and log1[26][0] < log1[25][0]   # the replaced bodies (earlier t0) were found
    assert all(np.array_equal(s1[k], s0[k]) for k in s1)


def test_hot_path_calls_between_blocks_do_not_disturb_the_loop(oracle):
    """The block loop and the hot path share a context (predicted records, the deferred predictor, selection minima,
    speculative descriptors).  nb_predict_all + nb_regular on arbitrary blocks -- small (fused predictor), large
    (records, Morton reordering) -- and nb_get_predicted between block steps must leave the integration untouched:
    the state after the mixed sequence equals the state after the block steps alone, bit for bit, and the
    interleaved nb_regular results still match the oracle at the time they were asked for."""
    import paper_1504_03687_b200 as nb
    from tests import parity
    cfg = nbgen.make_config(3, N=20000, n_i=16)
    N, cap = cfg["N"], cfg["cap"]
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    t0 = np.floor(0.3 / dt) * dt
    eta, dt_max = 0.02, 2.0**-6

    def run(mixed):
        ctx = nb.nb_open(N, cap)
        nb.nb_set_j(ctx, *(_dev(a) for a in (cfg["m"], cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], t0)))
        ctx.set_steps(_dev(dt))
        log = []
        for b in range(30):
            log.append(ctx.block_step(None, eta, dt_max))
            if mixed and b % 3 == 1:
                n_i = (7, 100, 5000)[(b // 3) % 3]
                idx, h2 = nbgen.active_block(cfg, n_i)
                t_q = log[-1][0] + 2.0**-20
                ctx.predict_all(t_q)
                got = parity.to_numpy(ctx.regular_alloc(_dev(idx, torch.int32), _dev(h2)))
                ctx.synchronize()
                s = _state(ctx, with_steps=False)
                xp, vp = oracle.predict(s["x0"], s["v0"], s["a0"], s["j0"], s["t0"], t_q)
                ref = parity.oracle_reference(oracle, s["m"], xp, vp, idx, h2, cap)
                parity.compare(got, ref, cap)
        log.append(ctx.run_blocks(None, eta, dt_max, t_stop=1.0e9, max_blocks=20))
        out = _state(ctx)
        ctx.close()
        return log, out

    log0, s0 = run(False)
    log1, s1 = run(True)
    assert log0 == log1
    assert all(np.array_equal(s0[k], s1[k]) for k in s0)


@pytest.mark.parametrize("variant", [0, 1, 4])
def test_block_loops_with_a_forced_kernel_variant_follow_the_oracle(variant):
    """NB_TUNE_FORCE_VARIANT inside nb_block_step / nb_run_blocks.  Variants 0 and 1 have no fused form and variant 4
    holds 32 particles per CTA, so a small block's speculative chain (block time known on the device only) would have
    to take the records route, which predicts to the HOST's time: the loop must not speculate there (round-2 advisor
    finding: it did, and integrated with forces evaluated at t = 0).  40 blocks in lockstep with the oracle, then the
    same 40 blocks by nb_run_blocks: bit-identical to the single calls."""
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(3, N=12000)
    N = cfg["N"]
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    st = dict(x0=cfg["x0"].copy(), v0=cfg["v0"].copy(), a0=cfg["a0"].copy(), j0=cfg["j0"].copy(),
              t0=np.floor(0.3 / dt) * dt, dt=dt.copy())
    start = {k: v.copy() for k, v in st.items()}
    m = cfg["m"]
    eta, dt_max, K = 0.02, 2.0**-6, 40

    def fresh():
        ctx = nb.nb_open(N, 8)
        nb.nb_set_j(ctx, *(_dev(a) for a in (m, start["x0"], start["v0"], start["a0"], start["j0"], start["t0"])))
        ctx.set_steps(_dev(start["dt"]))
        ctx.tune("force_variant", variant)
        return ctx

    ctx = fresh()
    sizes, flips = [], 0
    for b in range(K):
        t, n = ctx.block_step(None, eta, dt_max)
        assert ctx.info("last_variant") == variant
        t_ref, act, _ = _oracle_block(st, m, eta, dt_max)
        assert t == t_ref and n == act.size, (b, t, t_ref, n, act.size)
        assert np.array_equal(ctx.get_block(n)["idx_act"].cpu().numpy(), act), b
        sizes.append(n)
        g_dt = _state(ctx)["dt"]
        diff = np.flatnonzero(g_dt != st["dt"])
        assert np.isin(diff, act).all()
        flips += diff.size
        st["dt"][diff] = g_dt[diff]
    got = _state(ctx)
    hits = ctx.info("spec_hits")
    print("forced variant", variant, "sizes min/median/max", min(sizes), int(np.median(sizes)), max(sizes), "flips", flips,
          "speculative hits", hits)
    assert min(sizes) <= 32                                          # blocks that WOULD have been speculated
    if variant < 2:
        assert hits == 0 and ctx.info("spec_misses") == 0            # no speculative chain was ever enqueued
    assert flips <= max(2, int(1e-3 * sum(sizes)))
    assert np.array_equal(got["t0"], st["t0"])
    assert np.abs(got["x0"] - st["x0"]).max() < 5e-9 and np.abs(got["v0"] - st["v0"]).max() < 6e-6
    scale = np.linalg.norm(st["a0"], axis=1)
    assert np.max(np.linalg.norm(got["a0"] - st["a0"], axis=1) / scale) <= 1e-5
    ctx.close()
    ctx = fresh()
    t2, blocks, steps = ctx.run_blocks(None, eta, dt_max, max_blocks=K)
    assert blocks == K and steps == sum(sizes)
    run = _state(ctx)
    for key in got:
        assert np.array_equal(run[key], got[key]), key
    ctx.close()


def test_get_block_copies_no_more_than_the_caller_has_room_for():
    """nb_get_block(n_cap, ...): min(n_cap, size of the last block) rows (round-2 advisor finding: it used to copy the
    block's size whatever the caller had allocated); NB_INFO_LAST_BLOCK_N tells that size after nb_run_blocks."""
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(2, N=20000, n_i=16)
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    ctx = nb.nb_open(cfg["N"], 8)
    nb.nb_set_j(ctx, *(_dev(cfg[k]) for k in ("m", "x0", "v0", "a0", "j0")), _dev(np.floor(0.3 / dt) * dt))
    ctx.set_steps(_dev(dt))
    t, n = ctx.block_step(None, 0.02, 2.0**-6)
    assert n > 8 and ctx.info("last_block_n") == n
    full = ctx.get_block(n)
    half = n // 2
    guard = torch.full((n, 3), 7.0, dtype=torch.float64, device="cuda")      # room for n, told half
    idx = torch.full((n,), -7, dtype=torch.int32, device="cuda")
    from paper_1504_03687_b200.binding import _check, _vp
    _check(ctx._lib.nb_get_block(ctx._ctx, half, _vp(idx.data_ptr()), _vp(guard.data_ptr()), _vp(), _vp(), _vp(), _vp(), _vp()),
           "nb_get_block", ctx._ctx)
    ctx.synchronize()
    assert torch.equal(idx[:half], full["idx_act"][:half]) and bool((idx[half:] == -7).all())
    assert torch.equal(guard[:half], full["acc"][:half]) and bool((guard[half:] == 7.0).all())
    more = ctx.get_block(n + 100)                                            # more room than rows: n rows copied
    assert torch.equal(more["idx_act"][:n], full["idx_act"])
    tt, blocks, steps = ctx.run_blocks(None, 0.02, 2.0**-6, max_blocks=3)
    last = ctx.info("last_block_n")
    assert blocks == 3 and 0 < last <= steps
    st = _state(ctx)
    blk = ctx.get_block(last)["idx_act"].cpu().numpy()
    assert np.all(st["t0"][blk] == st["t0"].max()) and (st["t0"] == st["t0"].max()).sum() == last
    ctx.close()


@pytest.mark.parametrize("grid,chunks", [(1, 1), (3, 1), (4, 0)])
def test_selection_with_several_chunks_per_cta_selects_the_same_blocks(grid, chunks):
    """The scatter kernel's look-back (a chunk waits for the counts of the chunks before it) is safe because the grid
    never exceeds what the device holds at once; beyond that a CTA walks several chunks in ascending order (round-2
    advisor / verdict finding: it used to rest on dispatch order from ~2.4M bodies up).  NB_TUNE_SELECT_GRID forces
    that route at N = 20000 (10 chunks on 1, 3 or 4 CTAs): same blocks, bit-identical state."""
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(3, N=20000, n_i=16)
    N = cfg["N"]
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    t0 = np.floor(0.3 / dt) * dt
    eta, dt_max = 0.02, 2.0**-6

    def run(cap):
        ctx = nb.nb_open(N, 8)
        ctx.tune("select_chunks", chunks)
        ctx.tune("select_grid", cap)
        assert ctx.info("select_grid") == cap
        nb.nb_set_j(ctx, *(_dev(a) for a in (cfg["m"], cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], t0)))
        ctx.set_steps(_dev(dt))
        log = [ctx.block_step(None, eta, dt_max) for _ in range(10)]
        log.append(ctx.run_blocks(None, eta, dt_max, t_stop=1.0e9, max_blocks=40))
        blk = ctx.get_block(ctx.info("last_block_n"))["idx_act"].cpu().numpy()
        out = _state(ctx)
        ctx.close()
        return log, blk, out

    log_c, blk_c, s_c = run(grid)
    log_0, blk_0, s_0 = run(0)
    assert log_c == log_0 and np.array_equal(blk_c, blk_0) and np.all(np.diff(blk_c) > 0)
    assert all(np.array_equal(s_c[k], s_0[k]) for k in s_c)


def test_two_level_selection_with_several_chunks_per_cta():
    """The same for the two-level loop, whose scatter kernel also lists the bodies due for a regular step."""
    import paper_1504_03687_b200 as nb
    N, cap = 12000, 64
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    from scipy.spatial import cKDTree
    d, _ = cKDTree(x).query(x, k=13)
    h2 = (d[:, 12] * 1.0001) ** 2
    runs = []
    for grid in (2, 0):
        ctx = nb.nb_open(N, cap)
        z3 = np.zeros((N, 3))
        nb.nb_set_j(ctx, _dev(m), _dev(x), _dev(v), _dev(z3), _dev(z3), _dev(np.zeros(N)))
        ctx.tune("select_grid", grid)
        assert ctx.ac_init(0.0, _dev(h2), 0.01, 2.0**-4) == 0
        res = ctx.ac_run(0.01, 0.02, 2.0**-4, max_blocks=120)
        st = {k: v_.cpu().numpy() for k, v_ in ctx.get_state(True).items()}
        st.update({k: v_.cpu().numpy() for k, v_ in ctx.ac_get(False).items() if k not in ("idx_act", "idx_reg")})
        runs.append((res, st))
        ctx.close()
    assert runs[0][0] == runs[1][0] and runs[0][0][3] > 0            # regular steps were taken
    for k in runs[0][1]:
        assert np.array_equal(runs[0][1][k], runs[1][1][k]), k


def test_block_selection_at_five_million_bodies():
    """N = 5,000,000: 2442 selection chunks, about twice what a B200 holds at once (148 SMs x 8 CTAs), so every CTA of the
    capped grid walks two or three chunks.  Three blocks; each block's members must be exactly {j : t0 + dt = min}
    computed from the state the library held before the step (the definition), ascending."""
    import paper_1504_03687_b200 as nb
    N = 5_000_000
    rng = np.random.default_rng(11)
    x = rng.standard_normal((N, 3))
    v = 0.5 * rng.standard_normal((N, 3))
    m = np.full(N, 1.0 / N)
    z3 = np.zeros((N, 3))
    levels = 8 + np.minimum(rng.geometric(0.55, N) - 1, 16)          # deep levels hold few bodies
    dt = 2.0 ** -levels.astype(np.float64)
    ctx = nb.nb_open(N, 8)
    nb.nb_set_j(ctx, _dev(m), _dev(x), _dev(v), _dev(z3), _dev(z3), _dev(np.zeros(N)))
    ctx.set_steps(_dev(dt))
    t0 = np.zeros(N)
    sizes = []
    for b in range(3):
        t, n = ctx.block_step(None, 0.02, 2.0**-6)
        due = np.flatnonzero(t0 + dt == (t0 + dt).min())
        assert t == (t0 + dt).min() and n == due.size
        assert np.array_equal(ctx.get_block(n)["idx_act"].cpu().numpy(), due)
        sizes.append(n)
        st = ctx.get_state(True)
        t0, dt = st["t0"].cpu().numpy(), st["dt"].cpu().numpy()
        del st
        assert np.all(t0[due] == t)
    print("5M-body selection: block sizes", sizes, "chunks", (N + 2047) // 2048)
    assert 0 < min(sizes) and len(set(np.asarray(due) // 2048)) > 1
    ctx.close()
