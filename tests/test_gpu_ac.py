"""Two-level Ahmad-Cohen stepping on the GPU (nb_ac_init / nb_ac_step, readings R33-R38) against
oracle/hermite_ac.py on the same seeded inputs.  Needs a B200."""
import numpy as np
import pytest

import nbgen
from oracle import hermite_ac as AC

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def _radii(x, k):
    if x.shape[0] > 4096:                      # (a library routine, not the oracle: k-th neighbour distance)
        from scipy.spatial import cKDTree
        d, _ = cKDTree(x).query(x, k=k + 1)
        return d[:, k] ** 2 * 1.002
    d2 = ((x[:, None, :] - x[None, :, :]) ** 2).sum(-1)
    return np.sort(d2, axis=1)[:, k] * 1.002


def _open(m, x, v, cap):
    import paper_1504_03687_b200 as nb
    N = m.shape[0]
    ctx = nb.nb_open(N, cap)
    z3, z1 = np.zeros((N, 3)), np.zeros(N)
    nb.nb_set_j(ctx, _dev(m), _dev(x), _dev(v), _dev(z3), _dev(z3), _dev(z1))
    return ctx


def _gpu_state(ctx, lists=False):
    st = {k: v.cpu().numpy() for k, v in ctx.get_state(True).items()}
    st.update({k: v.cpu().numpy() for k, v in ctx.ac_get(lists).items()})
    return st


def _rel(a, b):
    s = np.linalg.norm(b, axis=1)
    return np.max(np.linalg.norm(a - b, axis=1) / np.where(s > 0, s, 1.0))


@pytest.mark.parametrize("N,cap,knb,nblocks", [(1024, 128, 16, 300), (12000, 64, 12, 60)])
def test_ac_start_and_blocks_in_lockstep_with_the_oracle(oracle, N, cap, knb, nblocks):
    """N = 1024: 300 blocks; N = 12000: the j-range spans 47 tiles and six selection chunks (one ragged), 60 blocks."""
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    h2 = _radii(x, knb)
    eta_I, eta_R, eta_s, dt_max = 0.01, 0.02, 0.01, 2.0**-4
    st = AC.start(oracle, m, x, v, h2, cap, eta_s, dt_max)
    ctx = _open(m, x, v, cap)
    assert ctx.ac_init(0.0, _dev(h2), eta_s, dt_max) == 0
    g = _gpu_state(ctx, lists=True)
    assert np.array_equal(g["nnb"], st["nnb"])
    for i in range(N):
        assert np.array_equal(g["nblist"][i, :g["nnb"][i]], st["list"][i, :st["nnb"][i]])
    assert _rel(g["aI"], st["aI"]) < 1e-12 and _rel(g["jI"], st["jI"]) < 1e-11       # FP64 neighbour force
    assert _rel(g["aR"], st["aR"]) < 1e-5 and _rel(g["jR"], st["jR"]) < 1e-4         # FP32 pair arithmetic
    assert _rel(g["a0"], st["a0"]) < 1e-5
    flips = int((g["dt"] != st["dtI"]).sum() + (g["dtR"] != st["dtR"]).sum())
    st["dtI"], st["dtR"] = g["dt"].copy(), g["dtR"].copy()                            # adopt flipped decisions
    isteps, rsteps, pure_irr = 0, 0, 0
    for b in range(nblocks):
        t, n, nr = ctx.ac_step(eta_I, eta_R, dt_max)
        t_ref, act, reg = AC.block_step(oracle, m, st, h2, cap, eta_I, eta_R, dt_max)
        g = _gpu_state(ctx)
        assert t == t_ref and n == act.size and nr == reg.size, (b, t, t_ref, n, act.size, nr, reg.size)
        assert np.array_equal(g["idx_act"][:n], act) and np.array_equal(g["idx_reg"][:nr], reg)
        isteps += n; rsteps += nr; pure_irr += int(nr == 0)
        dI, dR = np.flatnonzero(g["dt"] != st["dtI"]), np.flatnonzero(g["dtR"] != st["dtR"])
        assert np.isin(dI, act).all() and np.isin(dR, reg).all()
        flips += dI.size + dR.size
        st["dtI"][dI] = g["dt"][dI]; st["dtR"][dR] = g["dtR"][dR]
        assert np.all(g["dt"] <= g["dtR"])
    g = _gpu_state(ctx, lists=True)
    print("AC lockstep: blocks", nblocks, "irregular steps", isteps, "regular steps", rsteps, "blocks without a regular step",
          pure_irr, "flips", flips, "max |dx|", np.abs(g["x0"] - st["x0"]).max())
    assert pure_irr > nblocks // 3 and (rsteps > 0 or N > 1024)
    assert flips <= max(3, int(2e-3 * (isteps + rsteps)))
    assert np.array_equal(g["t0"], st["t0"]) and np.array_equal(g["tR"], st["tR"])
    assert np.abs(g["x0"] - st["x0"]).max() < 1e-9 and np.abs(g["v0"] - st["v0"]).max() < 1e-7
    assert _rel(g["aI"], st["aI"]) < 1e-7 and _rel(g["aR"], st["aR"]) < 1e-5
    same_lists = sum(np.array_equal(g["nblist"][i, :g["nnb"][i]], st["list"][i, :st["nnb"][i]]) for i in range(N))
    assert same_lists >= N - 2                                   # (a band pair may be classified differently)
    ctx.close()


def test_ac_without_neighbours_is_the_single_level_block_step_on_the_gpu():
    """Every h2 = 0: no lists, dtI = dtR, and nb_ac_step must reproduce nb_block_step (same force kernel, the
    corrector written as irregular corrector + regular correction): same blocks, same steps, states to rounding."""
    import paper_1504_03687_b200 as nb
    N = 2048
    cfg = nbgen.make_config(2, N=N, n_i=16)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    eta, eta_s, dt_max = 0.02, 0.02, 2.0**-5
    a = _open(m, x, v, 8)
    assert a.ac_init(0.0, _dev(np.zeros(N)), eta_s, dt_max) == 0
    ga = _gpu_state(a)
    b = nb.nb_open(N, 8)
    z1 = np.zeros(N)
    nb.nb_set_j(b, _dev(m), _dev(x), _dev(v), _dev(ga["a0"]), _dev(ga["j0"]), _dev(z1))
    b.init_steps(eta_s, dt_max)
    for blk in range(60):
        ta, na, nra = a.ac_step(0.005, eta, dt_max)
        tb, nb_ = b.block_step(None, eta, dt_max)
        assert ta == tb and na == nb_ == nra, (blk, ta, tb, na, nb_, nra)
    ga = _gpu_state(a)
    gb = {k: v.cpu().numpy() for k, v in b.get_state(True).items()}
    assert np.array_equal(ga["dt"], gb["dt"]) and np.array_equal(ga["dtR"], gb["dt"]) and np.array_equal(ga["t0"], gb["t0"])
    # the two correctors group the same terms differently (x' + (A + B) against ((x' + A) + B)): a 1e-16 difference
    # in x now and then flips an FP32 rounding inside the next force sum (1e-7 of a pair term), so the two runs agree
    # to the noise of the FP32 force, ~1e-7 |a| dt^2, not to FP64 rounding; a missing correction term would be ~1e-5
    assert np.abs(ga["x0"] - gb["x0"]).max() < 1e-10 and np.abs(ga["v0"] - gb["v0"]).max() < 1e-8
    assert not ga["aI"].any() and ga["nnb"].sum() == 0
    a.close(); b.close()


def test_ac_run_conserves_energy_and_overflow_is_reported(oracle):
    import paper_1504_03687_b200 as nb
    N, cap = 1024, 128
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    h2 = _radii(x, 16)
    eta_I, eta_R, eta_s, dt_max, t_end = 0.01, 0.02, 0.01, 2.0**-4, 0.125

    def energy(xx, vv):
        pot = oracle.regular(m, xx, vv, np.arange(N, dtype=np.int32), np.zeros(N), 8, want_list=False)["pot"]
        return 0.5 * (m * (vv * vv).sum(1)).sum() + 0.5 * (m * pot).sum()

    e0 = energy(x, v)
    ctx = _open(m, x, v, cap)
    ctx.ac_init(0.0, _dev(h2), eta_s, dt_max)
    t, blocks, isteps, rsteps = ctx.ac_run(eta_I, eta_R, dt_max, t_stop=t_end, max_blocks=100)      # the loop inside the library
    assert blocks == 100 and t < t_end
    t, b2, i2, r2 = ctx.ac_run(eta_I, eta_R, dt_max, t_stop=t_end)
    assert t > t_end and b2 > 0
    blocks += b2; isteps += i2; rsteps += r2
    assert ctx.ac_run(eta_I, eta_R, dt_max, t_stop=t_end)[1:] == (0, 0, 0)                        # nothing left before t_end
    g = _gpu_state(ctx)
    assert np.all(g["t0"] == t_end) and np.all(g["tR"] == t_end)
    e1 = energy(g["x0"], g["v0"])
    ref = AC.integrate(oracle, m, x, v, h2, cap, t_end, eta_I, eta_R, eta_s, dt_max)
    print("AC run on the GPU: blocks", blocks, "irregular steps", isteps, "regular steps", rsteps, "dE/E", (e1 - e0) / e0,
          "oracle", ref["blocks"], ref["irregular_steps"], ref["regular_steps"], "max |dx| vs oracle", np.abs(g["x0"] - ref["x0"]).max())
    assert abs((e1 - e0) / e0) < 5e-6
    assert isteps > 2 * rsteps > 0
    assert abs(isteps - ref["irregular_steps"]) <= 0.01 * ref["irregular_steps"]
    assert np.abs(g["x0"] - ref["x0"]).max() < 1e-5
    ctx.close()
    # radii that hold more bodies than the lists can: an error of the start-up, nothing is integrated
    ctx = _open(m, x, v, 8)
    with pytest.raises(nb.NbregError) as e:
        ctx.ac_init(0.0, _dev(h2), eta_s, dt_max)
    assert e.value.code == nb.NB_EOVERFLOW
    with pytest.raises(nb.NbregError) as e:
        ctx.ac_step(eta_I, eta_R, dt_max)
    assert e.value.code == nb.NB_ESTATE
    ctx.close()
    # a call that advances the state outside the two-level scheme ends it until the next nb_ac_init
    ctx = _open(m, x, v, cap)
    ctx.ac_init(0.0, _dev(h2), eta_s, dt_max)
    ctx.ac_step(eta_I, eta_R, dt_max)
    ctx.block_step(None, eta_R, dt_max)
    with pytest.raises(nb.NbregError) as e:
        ctx.ac_step(eta_I, eta_R, dt_max)
    assert e.value.code == nb.NB_ESTATE
    ctx.close()


def test_batched_loops_equal_block_by_block_stepping():
    """nb_ac_run / nb_run_blocks enqueue batches of blocks without the host in between (speculative chains, device
    stall flag, adaptive batch size).  Whatever the batching, the kernels and their order are the same: the state
    after K blocks must be BIT-identical to K single calls, with and without speculation, and with the neighbour
    force of the host-driven blocks (start-up, regular steps, large blocks) gathering predicted 64 B records
    (NB_TUNE_IRR_PRED_MIN = 1) instead of predicting every listed neighbour from its state line."""
    import paper_1504_03687_b200 as nb
    N, cap = 3000, 96
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    h2 = _radii(x, 12)
    eta_I, eta_R, eta_s, dt_max = 0.01, 0.02, 0.01, 2.0**-4
    runs = {}
    for mode in ("steps", "run", "run_nospec", "run_pred"):
        ctx = _open(m, x, v, cap)
        if mode == "run_nospec":
            ctx.tune("speculate", 0)
        if mode == "run_pred":               # every host-driven neighbour-force launch gathers predicted records
            ctx.tune("irr_pred_min", 1)
        ctx.ac_init(0.0, _dev(h2), eta_s, dt_max)
        K, ni, nr = 260, 0, 0
        if mode == "steps":
            for _ in range(K):
                t, a, b = ctx.ac_step(eta_I, eta_R, dt_max)
                ni += a; nr += b
        else:
            t, blocks, ni, nr = ctx.ac_run(eta_I, eta_R, dt_max, max_blocks=100)
            t, b2, i2, r2 = ctx.ac_run(eta_I, eta_R, dt_max, max_blocks=K - 100)
            assert blocks == 100 and b2 == K - 100
            ni += i2; nr += r2
        runs[mode] = (_gpu_state(ctx, lists=True), t, ni, nr, ctx.info("spec_hits"), ctx.info("spec_misses"))
        ctx.close()
    ref, t, ni, nr, hits, misses = runs["steps"]
    assert hits > 100 and nr > 0
    print("batched loops: irregular steps", ni, "regular steps", nr, "speculation hits / misses: steps", (hits, misses),
          "run", runs["run"][4:], "run without speculation", runs["run_nospec"][4:])
    assert runs["run_nospec"][4] == 0
    for mode in ("run", "run_nospec", "run_pred"):
        g, t2, ni2, nr2 = runs[mode][:4]
        assert (t2, ni2, nr2) == (t, ni, nr)
        for key in ("x0", "v0", "a0", "j0", "t0", "dt", "aI", "jI", "aR", "jR", "tR", "dtR", "nnb"):
            assert np.array_equal(g[key], ref[key]), (mode, key)
        for i in range(N):
            assert np.array_equal(g["nblist"][i, :g["nnb"][i]], ref["nblist"][i, :ref["nnb"][i]])
    # the single-level loop likewise
    states = []
    for mode in ("steps", "run"):
        ctx = nb.nb_open(N, 8)
        nb.nb_set_j(ctx, _dev(m), _dev(x), _dev(v), _dev(ref["a0"] * 0 + runs["steps"][0]["a0"]), _dev(runs["steps"][0]["j0"]),
                    _dev(np.zeros(N)))
        ctx.init_steps(eta_s, dt_max)
        if mode == "steps":
            tot = 0
            for _ in range(150):
                tt, n = ctx.block_step(None, 0.02, dt_max)
                tot += n
        else:
            tt, blocks, tot = ctx.run_blocks(None, 0.02, dt_max, max_blocks=150)
            assert blocks == 150
        states.append(({k: v_.cpu().numpy() for k, v_ in ctx.get_state(True).items()}, tt, tot))
        ctx.close()
    assert states[0][1:] == states[1][1:]
    for key in states[0][0]:
        assert np.array_equal(states[0][0][key], states[1][0][key]), key


def test_ac_overflow_in_mid_run_is_reported_at_the_same_block_as_the_oracle(oracle):
    """Lists sized exactly for the start-up state: as the cluster moves some body collects one neighbour too many at
    a regular step.  The library must return NB_EOVERFLOW for the very block at which the oracle raises, BEFORE
    correcting anything (the state is untouched and the same call fails again), reading R38."""
    import paper_1504_03687_b200 as nb
    N = 512
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    h2 = _radii(x, 10)
    eta_I, eta_R, eta_s, dt_max = 0.01, 0.02, 0.01, 2.0**-4
    probe = AC.start(oracle, m, x, v, h2, N, eta_s, dt_max)
    cap = int(probe["nnb"].max())                      # no slack at all
    st = AC.start(oracle, m, x, v, h2, cap, eta_s, dt_max)
    ctx = _open(m, x, v, cap)
    assert ctx.ac_init(0.0, _dev(h2), eta_s, dt_max) == 0
    g = _gpu_state(ctx)
    st["dtI"], st["dtR"] = g["dt"].copy(), g["dtR"].copy()
    for b in range(4000):
        before = _gpu_state(ctx)
        try:
            t_ref, act, reg = AC.block_step(oracle, m, st, h2, cap, eta_I, eta_R, dt_max)
            orc_raised = False
        except OverflowError:
            orc_raised = True
        try:
            t, n, nr = ctx.ac_step(eta_I, eta_R, dt_max)
            gpu_raised = False
        except nb.NbregError as e:
            assert e.code == nb.NB_EOVERFLOW
            gpu_raised = True
        assert orc_raised == gpu_raised, (b, orc_raised, gpu_raised)
        if gpu_raised:
            after = _gpu_state(ctx)
            for key in ("x0", "v0", "a0", "j0", "t0", "dt", "aI", "aR", "tR", "dtR", "nnb"):
                assert np.array_equal(before[key], after[key]), key            # nothing was corrected
            with pytest.raises(nb.NbregError) as e2:
                ctx.ac_step(eta_I, eta_R, dt_max)                               # the same block, the same error
            assert e2.value.code == nb.NB_EOVERFLOW
            print("overflow reported at block", b, "cap", cap)
            # ---- recovery (round-2 advisor finding: there was none).  Re-initialising in mid-run is refused ...
            with pytest.raises(nb.NbregError) as e3:
                ctx.ac_init(0.0, _dev(h2), eta_s, dt_max)
            assert e3.value.code == nb.NB_ESTATE
            still = _gpu_state(ctx)
            for key in ("x0", "v0", "a0", "j0", "t0", "dt", "aI", "aR", "tR", "dtR", "nnb"):
                assert np.array_equal(before[key], still[key]), key
            # ... the library names the regular steps it attempted and the true size of each new list ...
            f_idx, f_nnb = (a.cpu().numpy() for a in ctx.ac_get_failed())
            t_blk = (before["t0"] + before["dt"]).min()
            due = np.flatnonzero((before["t0"] + before["dt"] == t_blk) & (before["tR"] + before["dtR"] == t_blk))
            assert np.array_equal(f_idx, due)
            xp, vp = oracle.predict(st["x0"], st["v0"], st["a0"], st["j0"], st["t0"], t_blk)
            true_nnb = oracle.regular(m, xp, vp, due, h2[due], N)["nnb"]
            assert np.array_equal(f_nnb, true_nnb) and (f_nnb > cap).any()
            # ... the caller shrinks those radii and the SAME block goes through, in step with the oracle given the same radii
            bad = f_nnb > cap
            h2 = h2.copy()
            h2[f_idx[bad]] *= (0.6 * cap / f_nnb[bad]) ** (2.0 / 3.0)
            ctx.ac_set_radii(_dev(f_idx[bad].astype(np.int32)), _dev(h2[f_idx[bad]]))
            for b2 in range(30):
                try:
                    t_ref, act, reg = AC.block_step(oracle, m, st, h2, cap, eta_I, eta_R, dt_max)
                    orc_raised = False
                except OverflowError:
                    orc_raised = True
                try:
                    t, n, nr = ctx.ac_step(eta_I, eta_R, dt_max)
                    gpu_raised = False
                except nb.NbregError as e4:
                    assert e4.code == nb.NB_EOVERFLOW
                    gpu_raised = True
                assert orc_raised == gpu_raised, (b2, orc_raised, gpu_raised)
                if gpu_raised:
                    assert b2 > 0                       # the redone block itself must pass; a later one may overflow again
                    break
                assert t == t_ref and n == act.size and nr == reg.size, (b2, t, t_ref, n, act.size, nr, reg.size)
                if b2 == 0:
                    assert t == t_blk and np.array_equal(reg, due)
                    assert ctx.ac_get_failed()[0].numel() == 0
                g = _gpu_state(ctx)
                dI, dR = np.flatnonzero(g["dt"] != st["dtI"]), np.flatnonzero(g["dtR"] != st["dtR"])
                st["dtI"][dI] = g["dt"][dI]; st["dtR"][dR] = g["dtR"][dR]
            g = _gpu_state(ctx)
            assert np.array_equal(g["t0"], st["t0"]) and np.array_equal(g["nnb"], st["nnb"])
            assert np.abs(g["x0"] - st["x0"]).max() < 1e-9 and np.abs(g["v0"] - st["v0"]).max() < 1e-7
            print("recovered: redone block with", int(bad.sum()), "shrunk radii, then", b2, "more blocks in step with the oracle")
            break
        g = _gpu_state(ctx)
        dI, dR = np.flatnonzero(g["dt"] != st["dtI"]), np.flatnonzero(g["dtR"] != st["dtR"])
        st["dtI"][dI] = g["dt"][dI]; st["dtR"][dR] = g["dtR"][dR]
    else:
        pytest.fail("no overflow within 4000 blocks: the test set-up does not exercise the error path")
    ctx.close()


def test_get_block_after_a_two_level_step_is_refused():
    """nb_get_block reads the single-level loop's buffers; after nb_ac_step they are stale (results: nb_ac_get)."""
    import paper_1504_03687_b200 as nb
    N, cap = 512, 64
    cfg = nbgen.make_config(1, N=N)
    m, x, v = cfg["m"], cfg["x0"], cfg["v0"]
    ctx = _open(m, x, v, cap)
    assert ctx.ac_init(0.0, _dev(_radii(x, 10)), 0.01, 2.0**-4) == 0
    t, n, nr = ctx.ac_step(0.01, 0.02, 2.0**-4)
    assert n > 0 and ctx.info("last_block_n") == 0
    with pytest.raises(nb.NbregError) as e:
        ctx.get_block(n)
    assert e.value.code == nb.NB_ESTATE
    ctx.close()
