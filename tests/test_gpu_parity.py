"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs (BASELINE.json tolerances; tests/parity.py implements the band rule).  Needs a B200."""
import numpy as np
import pytest

import nbgen
from tests import parity

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def open_ctx(cfg, cap=None):
    import paper_1504_03687_b200 as nb
    ctx = nb.nb_open(cfg["N"], cap or cfg["cap"])
    nb.nb_set_j(ctx, _dev(cfg["m"]), _dev(cfg["x0"]), _dev(cfg["v0"]), _dev(cfg["a0"]), _dev(cfg["j0"]),
                _dev(cfg["t0"]))
    nb.nb_predict_all(ctx, cfg["t"])
    return ctx


def gpu_regular(ctx, idx_i, h2_i):
    out = ctx.regular_alloc(_dev(idx_i, torch.int32), _dev(h2_i))
    ctx.synchronize()
    return parity.to_numpy(out)


def gpu_predicted(ctx):
    xp = torch.empty((ctx.N, 3), dtype=torch.float64, device="cuda")
    vp = torch.empty((ctx.N, 3), dtype=torch.float64, device="cuda")
    ctx.get_predicted(xp, vp)
    ctx.synchronize()
    return xp.cpu().numpy(), vp.cpu().numpy()


def check(oracle, ctx, cfg, idx_i=None, h2_i=None, cap=None, **kw):
    idx_i = cfg["idx_i"] if idx_i is None else idx_i
    h2_i = cfg["h2_i"] if h2_i is None else h2_i
    cap = cap or cfg["cap"]
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, idx_i, h2_i, cap)
    got = gpu_regular(ctx, idx_i, h2_i)
    return parity.compare(got, ref, cap, **kw), got, ref


def _config1(oracle):
    cfg = nbgen.make_config(1)
    tot = oracle.regular(cfg["m"], cfg["x0"], cfg["v0"], cfg["idx_i"], np.zeros(cfg["N"]), cfg["cap"])
    xp, _ = oracle.predict(cfg["x0"], cfg["v0"], tot["acc"], tot["jerk"], cfg["t0"], cfg["t"])
    return nbgen.finish_config1(cfg, tot["acc"], tot["jerk"], xp)


# ----------------------------------------------------------------------------- predictor (a1, a2)

def test_predictor_dyadic_bitwise(oracle):
    rng = np.random.default_rng(0)
    n = 1000                                         # ragged: not a multiple of the 256-body tile
    q = lambda s, b: rng.integers(-2 ** b, 2 ** b, size=s) / 2.0 ** 4
    x0, v0, a0, j0 = q((n, 3), 10), q((n, 3), 6), 2 * q((n, 3), 6), 6 * q((n, 3), 6)
    k = rng.integers(2, 5, size=n)
    t0 = 1.0 - 2.0 ** -k
    cfg = dict(N=n, cap=8, m=rng.integers(1, 2 ** 10, size=n) / 2.0 ** 20, x0=x0, v0=v0, a0=a0, j0=j0, t0=t0, t=1.0)
    ctx = open_ctx(cfg)
    xg, vg = gpu_predicted(ctx)
    xo, vo = oracle.predict(x0, v0, a0, j0, t0, 1.0)
    assert np.array_equal(xg, xo) and np.array_equal(vg, vo)


def test_predictor_general(oracle):
    cfg = nbgen.make_config(3, N=20000, n_i=64)
    ctx = open_ctx(cfg)
    xg, vg = gpu_predicted(ctx)
    xo, vo = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    # x is stored as an FP32 hi/lo pair (48 bits), v as FP32 (24 bits); errors are relative to the
    # size of the summed Taylor terms (a component may cancel to near zero)
    def scales(t):
        dt = np.abs(t - cfg["t0"])[:, None]
        sx = np.abs(cfg["x0"]) + np.abs(cfg["v0"]) * dt + np.abs(cfg["a0"]) * dt ** 2 / 2 + np.abs(cfg["j0"]) * dt ** 3 / 6
        sv = np.abs(cfg["v0"]) + np.abs(cfg["a0"]) * dt + np.abs(cfg["j0"]) * dt ** 2 / 2
        return sx, sv
    sx, sv = scales(cfg["t"])
    assert np.max(np.abs(xg - xo) / sx) < 2.0 ** -46
    assert np.max(np.abs(vg - vo) / sv) < 2.0 ** -23.9
    # backward prediction (t < t0) is the same polynomial
    import paper_1504_03687_b200 as nb
    nb.nb_predict_all(ctx, 0.5)
    xg, _ = gpu_predicted(ctx)
    xo, _ = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], 0.5)
    assert np.max(np.abs(xg - xo) / scales(0.5)[0]) < 2.0 ** -46


# ----------------------------------------------------------------------------- configs 1, 2 in full

def test_config1_all_active(oracle):
    cfg = _config1(oracle)
    ctx = open_ctx(cfg)
    rep, got, ref = check(oracle, ctx, cfg)
    assert rep["overflow_rows"] == 0 and got["nnb"].min() >= 48
    print("config1", rep)


def test_config2(oracle):
    cfg = nbgen.make_config(2)
    ctx = open_ctx(cfg)
    rep, got, _ = check(oracle, ctx, cfg)
    assert 60 < rep["nnb_mean"] < 140
    print("config2", rep)


# ----------------------------------------------------------------------------- every variant, ragged sizes

@pytest.mark.parametrize("n_i", [1, 2, 7, 8, 9, 16, 17, 31, 32, 33, 64, 100, 128, 257, 512, 1000, 3000])
def test_block_sizes_ragged_N(oracle, n_i):
    cfg = nbgen.make_config(3, N=9001, n_i=n_i)        # 9001 = 35 tiles + a tail of 41
    ctx = open_ctx(cfg)
    rep, _, _ = check(oracle, ctx, cfg)
    assert ctx.info("last_grid") >= 1


@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("jsplit", [1, 3, 36])
def test_forced_variant_and_split_agree(oracle, variant, jsplit):
    """Split-j vs single pass and every thread mapping: identical neighbour sets, sums equal to FP64
    rounding of the final reduction (SURVEY 8(c) 'split-j path'; P:117-119 consistency)."""
    cfg = nbgen.make_config(3, N=9001, n_i=300)
    ctx = open_ctx(cfg)
    base = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    ctx.tune("force_variant", variant)
    ctx.tune("force_jsplit", jsplit)
    got = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    assert ctx.info("last_variant") == variant and ctx.info("last_jsplit") == jsplit
    assert np.array_equal(got["nnb"], base["nnb"]) and np.array_equal(got["overflow"], base["overflow"])
    for k in range(300):
        c = min(got["nnb"][k], cfg["cap"])
        assert set(got["nblist"][k, :c].tolist()) == set(base["nblist"][k, :c].tolist())
    for key, tol in (("acc", 3e-6), ("jerk", 3e-5), ("pot", 3e-7)):
        sc = np.linalg.norm(base[key].reshape(300, -1), axis=1)
        d = np.linalg.norm((got[key] - base[key]).reshape(300, -1), axis=1)
        assert np.max(d / sc) < tol          # different FP32 tile partition, same pairs
    rep, _, _ = check(oracle, ctx, cfg)


def test_bitwise_reproducible(oracle):
    cfg = nbgen.make_config(2, N=30000, n_i=777)
    ctx = open_ctx(cfg)
    a = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    b = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    for key in ("acc", "jerk", "pot", "nnb", "overflow"):
        assert np.array_equal(a[key], b[key])
    for k in range(777):
        if a["nnb"][k] <= cfg["cap"]:       # an overflowed row holds ANY cap-sized subset (reading R10)
            assert set(a["nblist"][k, :a["nnb"][k]].tolist()) == set(b["nblist"][k, :b["nnb"][k]].tolist())


# ----------------------------------------------------------------------------- degenerate / edge cases

def test_total_force_h2_zero_and_momentum(oracle):
    cfg = nbgen.make_config(2, N=4096, n_i=4096)
    cfg["idx_i"] = np.arange(4096, dtype=np.int32)
    h2 = np.zeros(4096)
    h2[::3] = -1.0                                              # h2 <= 0: no neighbours
    ctx = open_ctx(cfg)
    rep, got, _ = check(oracle, ctx, cfg, h2_i=h2)
    assert got["nnb"].sum() == 0 and got["overflow"].sum() == 0
    f = (cfg["m"][:, None] * got["acc"]).sum(0)
    assert np.abs(f).max() < 1e-6 * np.abs(cfg["m"][:, None] * got["acc"]).sum()


def test_overflow_small_cap(oracle):
    cfg = nbgen.make_config(2, N=8192, n_i=500)
    for cap in (1, 8, 100):
        ctx = open_ctx(cfg, cap=cap)
        rep, got, ref = check(oracle, ctx, cfg, cap=cap)
        assert rep["overflow_rows"] > 0 or cap == 100
        if cap == 100:
            assert 0 < rep["overflow_rows"] < 500             # mixes overflowing and fitting rows


def test_king_core_overflow_small_blocks(oracle):
    cfg = nbgen.make_config(5, N=131072, n_i=512)
    # shrink-N version of config 5: rescale the floor so the core still straddles the cap
    ctx = open_ctx(cfg)
    for n_i in (32, 128, 512):
        idx, h2 = nbgen.active_block(cfg, n_i)
        rep, got, _ = check(oracle, ctx, cfg, idx_i=idx, h2_i=h2)
        print("king", n_i, rep)
    assert rep["overflow_rows"] > 0


def test_translation_invariance_far_from_origin(oracle):
    """Shift every position by (100,-50,25): FP32 position differencing would fail this; the hi/lo
    split must stay inside the tolerances."""
    cfg = nbgen.make_config(2, N=8192, n_i=256)
    cfg = dict(cfg)
    cfg["x0"] = cfg["x0"] + np.array([100.0, -50.0, 25.0])
    ctx = open_ctx(cfg)
    check(oracle, ctx, cfg)


@pytest.mark.parametrize("v_bulk", [(3.0, -1.0, 2.0), (50.0, 0.0, 0.0)])
def test_velocity_frame_shift(oracle, v_bulk):
    """All velocities shifted by a bulk velocity (a cluster on a galactic orbit, or a frame that is not the
    centre-of-mass frame).  The kernel keeps v as ONE FP32, so the velocity difference
    carries an absolute error of 2^-24 |v_bulk| and the jerk a relative error of about 6e-8 |v_bulk| / sigma;
    (3,-1,2) is 7 sigma, (50,0,0) is ~100 sigma (sigma ~ 0.5 in N-body units) -- the stated limit of the
    FP32 choice.  BASELINE.json's jerk tolerances (1e-4 max, 1e-5 rms) must hold at both; acc / pot / lists
    do not depend on v at all."""
    base_cfg = dict(nbgen.make_config(2, N=8192, n_i=256))
    base_cfg["t0"] = np.full(8192, base_cfg["t"])          # dt = 0: the predicted positions do not depend on v
    cfg = dict(base_cfg)
    cfg["v0"] = cfg["v0"] + np.array(v_bulk)
    rep, got, _ = check(oracle, open_ctx(cfg), cfg)
    print("velocity frame", v_bulk, rep)
    base = gpu_regular(open_ctx(base_cfg), cfg["idx_i"], cfg["h2_i"])
    for key in ("acc", "pot", "nnb", "overflow"):           # only the jerk sees the velocities
        assert np.array_equal(got[key], base[key]), key


def test_everyone_is_a_neighbour(oracle):
    cfg = nbgen.make_config(2, N=2000, n_i=64)
    ctx = open_ctx(cfg, cap=4096)
    rep, got, _ = check(oracle, ctx, cfg, h2_i=np.full(64, 1e6), cap=4096)
    assert np.all(got["nnb"] == 1999) and not got["acc"].any() and not got["pot"].any()


@pytest.mark.parametrize("N", [1, 2, 3, 37, 255, 256, 257, 513])
def test_degenerate_sizes_everybody_active(oracle, N):
    """The smallest problems: N = 1 (no pair at all: exact zeros), 2, 3, one ragged tile, exactly one tile, one
    tile + 1, two tiles + 1 -- everybody active, seeded uniform cube with random masses / velocities / steps, a
    radius that gives a few neighbours, cap 4 (some rows overflow).  By both routes (records; FP64 state with the
    predictor fused where the block is small enough) and with h2 = 0 (momentum: sum m a = 0)."""
    rng = np.random.default_rng(1000 + N)
    x0 = rng.uniform(-1, 1, (N, 3)); v0 = rng.normal(0, 0.3, (N, 3))
    a0 = rng.normal(0, 0.5, (N, 3)); j0 = rng.normal(0, 0.5, (N, 3))
    t0 = 1.0 - 2.0 ** -rng.integers(3, 9, N).astype(np.float64)
    m = rng.uniform(0.5, 1.5, N) / N
    cfg = dict(N=N, cap=4, m=m, x0=x0, v0=v0, a0=a0, j0=j0, t0=t0, t=1.0)
    idx = np.arange(N, dtype=np.int32)
    h2 = np.full(N, (0.9 * (8.0 / max(N, 2)) ** (1.0 / 3.0)) ** 2)        # ~3 neighbours each
    for fuse in (1, 0):
        ctx = open_ctx(cfg)
        ctx.tune("fuse_predict", fuse)
        rep, got, ref = check(oracle, ctx, cfg, idx_i=idx, h2_i=h2, cap=4)
        assert ctx.info("last_fused") == (1 if fuse and N <= 128 else 0)
        if N == 1:
            assert not got["acc"].any() and not got["jerk"].any() and got["pot"][0] == 0 and got["nnb"][0] == 0
        if N >= 37:
            assert got["nnb"].max() > 0
        rep0, got0, _ = check(oracle, ctx, cfg, idx_i=idx, h2_i=np.zeros(N), cap=4)
        assert got0["nnb"].sum() == 0
        if N > 1:
            f = (m[:, None] * got0["acc"]).sum(0)
            assert np.abs(f).max() < 2e-6 * np.abs(m[:, None] * got0["acc"]).sum()
        ctx.close()


def test_two_body_closed_form():
    import paper_1504_03687_b200 as nb
    cfg = dict(N=2, cap=4, m=np.array([1.0, 1.0]), x0=np.array([[0, 0, 0], [3.0, 4.0, 0]]),
               v0=np.array([[0, 0, 0], [1.0, 2.0, 2.0]]), a0=np.zeros((2, 3)), j0=np.zeros((2, 3)),
               t0=np.zeros(2), t=0.0)
    ctx = open_ctx(cfg)
    got = gpu_regular(ctx, np.array([0], np.int32), np.array([0.0]))
    np.testing.assert_allclose(got["acc"][0], [0.024, 0.032, 0.0], rtol=1e-6, atol=1e-9)
    np.testing.assert_allclose(got["jerk"][0], [-0.02368, -0.02624, 0.016], rtol=5e-6, atol=1e-9)
    assert abs(got["pot"][0] + 0.2) < 2e-7
    got = gpu_regular(ctx, np.array([0], np.int32), np.array([26.0]))      # partner inside h: exact zeros
    assert got["nnb"][0] == 1 and got["nblist"][0, 0] == 1 and not got["acc"].any() and got["pot"][0] == 0


def test_api_errors_and_noop():
    import paper_1504_03687_b200 as nb
    from paper_1504_03687_b200 import NbregError
    with pytest.raises(NbregError) as e:
        nb.nb_open(0, 8)
    assert e.value.code == nb.NB_EINVAL
    with pytest.raises(NbregError):
        nb.nb_open(16, 0)
    ctx = nb.nb_open(300, 8)
    with pytest.raises(NbregError) as e:
        nb.nb_predict_all(ctx, 1.0)
    assert e.value.code == nb.NB_ESTATE
    z = lambda *s: torch.zeros(*s, dtype=torch.float64, device="cuda")
    x = torch.rand(300, 3, dtype=torch.float64, device="cuda")
    nb.nb_set_j(ctx, z(300) + 1.0 / 300, x, z(300, 3), z(300, 3), z(300, 3), z(300))
    idx = torch.arange(4, dtype=torch.int32, device="cuda")
    with pytest.raises(NbregError) as e:
        ctx.regular_alloc(idx, z(4))
    assert e.value.code == nb.NB_ESTATE
    nb.nb_predict_all(ctx, 0.0)
    launches = ctx.info("kernel_launches")
    ctx.regular_alloc(idx[:0], z(0))                                       # n_i = 0: valid no-op
    assert ctx.info("kernel_launches") == launches
    out = ctx.regular_alloc(idx, z(4))
    ctx.synchronize()
    assert torch.isfinite(out["acc"]).all() and ctx.info("kernel_launches") == launches + 2
    assert ctx.info("sm_count") >= 100
    ctx.close()


def test_host_variants_equal_device_variants(oracle):
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(2, N=10000, n_i=400)
    ctx = open_ctx(cfg)
    dev = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    ctx2 = nb.nb_open(cfg["N"], cfg["cap"])
    ctx2.set_j_host(*(np.ascontiguousarray(cfg[k]) for k in ("m", "x0", "v0", "a0", "j0", "t0")))
    ctx2.predict_all(cfg["t"])
    n, cap = 400, cfg["cap"]
    out = dict(acc=np.empty((n, 3)), jerk=np.empty((n, 3)), pot=np.empty(n), nnb=np.empty(n, np.int32),
               nblist=np.full((n, cap), -1, np.int32), overflow=np.empty(n, np.int32))
    ctx2.regular_host(np.ascontiguousarray(cfg["idx_i"]), np.ascontiguousarray(cfg["h2_i"]), **out)
    for key in ("acc", "jerk", "pot", "nnb", "overflow"):
        assert np.array_equal(out[key], dev[key])
    for k in range(n):
        if dev["nnb"][k] <= cap:
            assert set(out["nblist"][k, :out["nnb"][k]].tolist()) == set(dev["nblist"][k, :dev["nnb"][k]].tolist())


def _host_out(n, cap):
    return dict(acc=np.empty((n, 3)), jerk=np.empty((n, 3)), pot=np.empty(n), nnb=np.empty(n, np.int32),
                nblist=np.full((n, cap), -1, np.int32), overflow=np.empty(n, np.int32))


@pytest.mark.parametrize("N,n_i", [(10000, 400), (140000, 300), (600000, 320)])
def test_step_host_pipelined_matches_oracle_and_separate_calls(oracle, N, n_i):
    """nb_step_host (chunked copies, per-chunk force launches, host-gathered i-state) against the oracle
    and against set_j + predict_all + regular on a second context: 1, 3 and 5 chunks, ragged last tile,
    active particles drawn from every chunk."""
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(2, N=N, n_i=n_i)
    cap = cfg["cap"]
    idx = np.ascontiguousarray(cfg["idx_i"]); h2 = np.ascontiguousarray(cfg["h2_i"])
    assert idx.min() < N // 16 and idx.max() > N // 2          # first and last chunk both hold active particles
    jst = [np.ascontiguousarray(cfg[k]) for k in ("m", "x0", "v0", "a0", "j0", "t0")]
    ctx = nb.nb_open(N, cap)
    out = _host_out(n_i, cap)
    ctx.step_host(*jst, cfg["t"], idx, h2, **out)
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, idx, h2, cap)
    rep = parity.compare(out, ref, cap)
    print("step_host", N, n_i, rep, "S_total", ctx.info("last_jsplit"))
    sep = gpu_regular(open_ctx(cfg), idx, h2)
    for key in ("nnb", "overflow"):
        assert np.array_equal(out[key], sep[key])
    for k in range(n_i):
        c = min(out["nnb"][k], cap)
        if out["nnb"][k] <= cap:
            assert np.array_equal(out["nblist"][k, :c], sep["nblist"][k, :c])      # sorted rows: identical
    # same pair terms; the FP32 tile sums of the WJ > 1 variants group differently when the j-range is
    # cut into chunks, the FP64 order differs always: agreement to FP32-sum rounding, far inside the tolerances
    for key, tol in (("acc", 5e-7), ("jerk", 5e-7), ("pot", 5e-7)):
        scale = np.abs(sep[key]).max()
        assert np.abs(out[key] - sep[key]).max() <= tol * scale
    # bitwise reproducible, and the context is left as after set_j + predict_all(t)
    out2 = _host_out(n_i, cap)
    ctx.step_host(*jst, cfg["t"], idx, h2, **out2)
    for key in ("acc", "jerk", "pot", "nnb", "overflow"):
        assert np.array_equal(out[key], out2[key])
    again = gpu_regular(ctx, idx, h2)
    for key in ("acc", "jerk", "pot", "nnb", "overflow"):
        assert np.array_equal(again[key], sep[key])
    ctx.close()


def test_step_host_errors_and_empty_block():
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(2, N=3000, n_i=10)
    jst = [np.ascontiguousarray(cfg[k]) for k in ("m", "x0", "v0", "a0", "j0", "t0")]
    ctx = nb.nb_open(3000, 64)
    out = _host_out(10, 64)
    bad = np.ascontiguousarray(cfg["idx_i"]).copy(); bad[3] = 3000
    with pytest.raises(nb.NbregError) as e:
        ctx.step_host(*jst, cfg["t"], bad, np.ascontiguousarray(cfg["h2_i"]), **out)
    assert e.value.code == nb.NB_EINVAL
    ctx.step_host(*jst, cfg["t"], np.empty(0, np.int32), None, None, None, None, None, None, None)   # = set_j + predict
    got = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    sep = gpu_regular(open_ctx(cfg, cap=64), cfg["idx_i"], cfg["h2_i"])
    assert np.array_equal(got["acc"], sep["acc"]) and np.array_equal(got["nnb"], sep["nnb"])
    ctx.close()


def test_j_sharding_three_shards_sum_to_the_whole(oracle):
    """three contiguous j-shards (three contexts, run one after the other on this GPU)
    each evaluate their part of the same active block with nb_regular_shard; the partial sums added and
    the list rows concatenated in shard order must equal the unsharded call and the oracle."""
    import paper_1504_03687_b200 as nb
    from paper_1504_03687_b200 import parallel as par
    cfg = nbgen.make_config(2, N=20011, n_i=333)
    N, cap, t = cfg["N"], cfg["cap"], cfg["t"]
    idx, h2 = _dev(cfg["idx_i"], torch.int32), _dev(cfg["h2_i"])
    whole = gpu_regular(open_ctx(cfg), cfg["idx_i"], cfg["h2_i"])
    b = par.shard_bounds(N, 3)
    assert b[0] == 0 and b[-1] == N and all(x % 256 == 0 for x in b[:-1]) and len(set(b)) == 4
    states = [{k: _dev(cfg[k][b[r]:b[r + 1]]) for k in par.STATE_KEYS} for r in range(3)]
    ist = sum(par.gather_istate(states[r], b[r], idx) for r in range(3))          # what the all-reduce would give
    assert (idx.cpu().numpy() >= b[2]).any() and (idx.cpu().numpy() < b[1]).any()  # active bodies in first and last shard
    parts = []
    for r in range(3):
        n_loc = b[r + 1] - b[r]
        ctx = nb.nb_open(n_loc, cap)
        nb.nb_set_j(ctx, *(states[r][k] for k in par.STATE_KEYS))
        ctx.set_j_offset(b[r])
        ctx.predict_all(t)
        part = dict(acc=torch.empty((333, 3), dtype=torch.float64, device="cuda"),
                    jerk=torch.empty((333, 3), dtype=torch.float64, device="cuda"),
                    pot=torch.empty(333, dtype=torch.float64, device="cuda"),
                    nnb=torch.empty(333, dtype=torch.int32, device="cuda"),
                    nblist=torch.full((333, cap), -1, dtype=torch.int32, device="cuda"),
                    overflow=torch.empty(333, dtype=torch.int32, device="cuda"))
        ctx.regular_shard(t, idx, ist.contiguous(), h2, **part)
        ctx.synchronize()
        parts.append(part)
        ctx.close()
    rows = torch.stack([p_["nblist"] for p_ in parts]); cnts = torch.stack([p_["nnb"].long() for p_ in parts])
    nblist, nnb, ovf = par.merge_list_rows(rows, cnts, cap)
    got = dict(acc=sum(p_["acc"] for p_ in parts), jerk=sum(p_["jerk"] for p_ in parts), pot=sum(p_["pot"] for p_ in parts),
               nnb=nnb, nblist=nblist, overflow=ovf)
    got = parity.to_numpy(got)
    assert np.array_equal(got["nnb"], whole["nnb"]) and np.array_equal(got["overflow"], whole["overflow"])
    for k in range(333):
        if got["nnb"][k] <= cap:         # (an overflowed row keeps ANY cap of its neighbours, R10)
            c = got["nnb"][k]
            assert np.array_equal(got["nblist"][k, :c], whole["nblist"][k, :c])   # shard order = ascending j
    for key in ("acc", "jerk", "pot"):
        assert np.abs(got[key] - whole[key]).max() <= 5e-7 * np.abs(whole[key]).max()
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], t)
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, cfg["idx_i"], cfg["h2_i"], cap)
    print("j-sharded x3", parity.compare(got, ref, cap))


# ----------------------------------------------------------------------------- full size (bench launch config)

_CFG4 = {}


def _config4(oracle):
    """Config 4 (N = 1,048,576), its context and the oracle's predicted state, built once per session."""
    if not _CFG4:
        cfg = nbgen.make_config(4)
        _CFG4["cfg"] = cfg
        _CFG4["ctx"] = open_ctx(cfg)
        _CFG4["pred"] = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    return _CFG4["cfg"], _CFG4["ctx"], _CFG4["pred"]


@pytest.mark.parametrize("n_i", [64, 128, 256, 512, 1024, 2048, 4096])
def test_config4_every_i_up_to_4096(oracle, n_i):
    """SURVEY 8(d) "Parity at 1M: all i for n_i <= 4096": every block size of config 4's sweep up to 4096
    at N = 1,048,576, every active particle against the oracle (each size has its own launch plan:
    variant, j-splits)."""
    cfg, ctx, (xp, vp) = _config4(oracle)
    idx, h2 = nbgen.active_block(cfg, n_i)
    got = gpu_regular(ctx, idx, h2)
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, idx, h2, cfg["cap"])
    rep = parity.compare(got, ref, cfg["cap"])
    print("config4 all-i", n_i, rep, "variant", ctx.info("last_variant"), "S", ctx.info("last_jsplit"))
    assert 100 < rep["nnb_mean"] < 220


@pytest.mark.parametrize("n_i", [8192, 16384, 32768, 65536])
def test_config4_sampled_4096_rows(oracle, n_i):
    """"for larger blocks a seeded subsample of 4096 i's" -- n_i = 8192 is the launch
    configuration bench.py times; nnb / overflow of the sampled rows are compared too."""
    cfg, ctx, (xp, vp) = _config4(oracle)
    idx, h2 = nbgen.active_block(cfg, n_i)
    got = gpu_regular(ctx, idx, h2)
    sel = np.sort(np.random.default_rng(n_i).choice(n_i, size=4096, replace=False))
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, idx[sel], h2[sel], cfg["cap"])
    rep = parity.compare({k: v[sel] for k, v in got.items()}, ref, cfg["cap"])
    print("config4 sample", n_i, rep, "variant", ctx.info("last_variant"), "S", ctx.info("last_jsplit"))
    assert np.all(np.isfinite(got["acc"])) and np.all(np.isfinite(got["jerk"])) and 100 < got["nnb"].mean() < 220


def test_full_size_step_host_bench_configuration(oracle):
    """The e2e leg of bench.py: nb_step_host at N = 1,048,576, n_i = 8192 with pinned host buffers; a
    seeded sample of the active particles against the oracle, everything against the separate calls."""
    import paper_1504_03687_b200 as nb
    cfg = _config4(oracle)[0]
    idx, h2 = nbgen.active_block(cfg, 8192)
    cap, n = cfg["cap"], 8192
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    jst = [pin(np.asarray(cfg[k], dtype=np.float64)) for k in ("m", "x0", "v0", "a0", "j0", "t0")]
    out = {k: torch.from_numpy(v).pin_memory() for k, v in _host_out(n, cap).items()}
    ctx = nb.nb_open(cfg["N"], cap)
    ctx.step_host(*jst, cfg["t"], pin(idx), pin(h2), **out)
    got = {k: v.numpy() for k, v in out.items()}
    sel = np.sort(np.random.default_rng(2).choice(n, size=4096, replace=False))      # 4096 rows
    xp, vp = _config4(oracle)[2]
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, idx[sel], h2[sel], cap)
    print("step_host config4 n_i=8192 sample", parity.compare({k: v[sel] for k, v in got.items()}, ref, cap),
          "S_total", ctx.info("last_jsplit"))
    sep = gpu_regular(ctx, idx, h2)
    assert np.array_equal(got["nnb"], sep["nnb"]) and np.array_equal(got["overflow"], sep["overflow"])
    fits = got["nnb"] <= cap
    m = np.arange(cap)[None, :] < got["nnb"][:, None]
    assert np.array_equal(got["nblist"][fits][m[fits]], sep["nblist"][fits][m[fits]])
    for key in ("acc", "jerk", "pot"):
        assert np.abs(got[key] - sep[key]).max() <= 1e-12 * np.abs(sep[key]).max()
    ctx.close()


def test_config5_full_size_king_core(oracle):
    """BASELINE.json configs[4] at its full size: N = 1,048,576 King W0 = 9, n_i = 32 / 128 / 512 of the
    innermost particles (split-j path at full N, rows above and below the 512 cap), every active
    particle checked by the oracle."""
    cfg = nbgen.make_config(5)
    ctx = open_ctx(cfg)
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    over = 0
    for n_i in cfg["sweep"]:
        idx, h2 = nbgen.active_block(cfg, n_i)
        got = gpu_regular(ctx, idx, h2)
        ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, idx, h2, cfg["cap"])
        rep = parity.compare(got, ref, cfg["cap"])
        print("config5 full", n_i, rep, "variant", ctx.info("last_variant"), "S", ctx.info("last_jsplit"))
        over = rep["overflow_rows"]
        assert ctx.info("last_jsplit") > 1                      # the j-range really is split
    assert 0 < over < 512                                       # mixes overflowing and fitting rows


@pytest.mark.parametrize("k,n_i", [(4, 3), (4, 8), (4, 16), (5, 8), (5, 16)])
def test_tiny_blocks_full_size(oracle, k, n_i):
    """The deep block levels hold a handful of particles: blocks of <= 16 take the j-packed
    variant with its lanes grouped along j (8 or 16 i-slots per warp instead of 32 padded ones).  N = 1,048,576,
    every active particle against the oracle, by both routes (FP64 state in with the predictor fused, and the
    predicted records); config 5's core rows overflow the 512 cap."""
    import paper_1504_03687_b200 as nb
    if k == 4:
        cfg, ctx, (xp, vp) = _config4(oracle)
    else:
        cfg = nbgen.make_config(5)
        ctx = open_ctx(cfg)
        xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    idx, h2 = nbgen.active_block(cfg, n_i)
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, idx, h2, cfg["cap"])
    out = {}
    for fused in (1, 0):
        nb.nb_predict_all(ctx, cfg["t"])                     # pending prediction: a small block fuses it
        ctx.tune("fuse_predict", fused)
        got = gpu_regular(ctx, idx, h2)
        assert ctx.info("last_fused") == fused and ctx.info("last_variant") == 4
        rep = parity.compare(got, ref, cfg["cap"])
        print("tiny block config", k, n_i, "fused" if fused else "records", rep, "S", ctx.info("last_jsplit"))
        out[fused] = got
    ctx.tune("fuse_predict", 1)
    assert np.array_equal(out[0]["nnb"], out[1]["nnb"]) and np.array_equal(out[0]["overflow"], out[1]["overflow"])
    if k == 5:
        assert out[1]["overflow"].sum() > 0
        ctx.close()


def test_config3_block_sweep_sampled(oracle):
    """BASELINE.json configs[2] at its full size (N = 262,144, 5 % binaries): the five block sizes of
    the sweep; the oracle checks every i up to n_i = 1024 and a seeded sample of 256 above."""
    cfg = nbgen.make_config(3)
    ctx = open_ctx(cfg)
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    for n_i in cfg["sweep"]:
        idx, h2 = nbgen.active_block(cfg, n_i)
        got = gpu_regular(ctx, idx, h2)
        sel = np.arange(n_i) if n_i <= 1024 else np.sort(np.random.default_rng(n_i).choice(n_i, 256, replace=False))
        ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, idx[sel], h2[sel], cfg["cap"])
        rep = parity.compare({k: v[sel] for k, v in got.items()}, ref, cfg["cap"])
        print("config3", n_i, rep, "variant", ctx.info("last_variant"), "S", ctx.info("last_jsplit"))
        assert np.all(np.isfinite(got["acc"])) and np.all(np.isfinite(got["jerk"]))


def test_config4_largest_block_sampled_and_block_independent(oracle):
    """N = 1,048,576, n_i = 131072 (the top of the sweep): a seeded sample of 4096 rows against the
    oracle, and -- a property that holds at any size -- a particle's result does not depend on the
    block it is computed in: the nested 8192-block gives the same counts, the same sets and sums equal
    up to the FP64 rounding of a different split (copies must not diverge)."""
    cfg, ctx, (xp, vp) = _config4(oracle)
    idx, h2 = nbgen.active_block(cfg, 131072)
    big = gpu_regular(ctx, idx, h2)
    sel = np.sort(np.random.default_rng(7).choice(131072, size=4096, replace=False))
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, idx[sel], h2[sel], cfg["cap"])
    rep = parity.compare({k: v[sel] for k, v in big.items()}, ref, cfg["cap"])
    print("config4 n_i=131072 sample", rep, "S", ctx.info("last_jsplit"))
    small = gpu_regular(ctx, idx[:8192], h2[:8192])
    assert np.array_equal(small["nnb"], big["nnb"][:8192])
    assert np.array_equal(small["overflow"], big["overflow"][:8192])
    for k in range(0, 8192, 17):
        c = min(small["nnb"][k], cfg["cap"])
        if small["nnb"][k] <= cfg["cap"]:
            assert set(small["nblist"][k, :c].tolist()) == set(big["nblist"][k, :c].tolist())
    # the two calls put a particle into different warps, i.e. different local origins: each evaluation carries a
    # position-difference error <= 1.8e-7 + 2.4e-7 G = 2.1e-6 at the default guard G = 8 for a
    # particle AT the guard; the bulk sits far inside it (measured max 8.6e-7), so two evaluations agree to a few 1e-6
    # at worst -- inside the 1e-5 / 1e-4 budget
    for key, tol in (("acc", 3e-6), ("jerk", 3e-5), ("pot", 3e-7)):
        a = small[key].reshape(8192, -1); b = big[key][:8192].reshape(8192, -1)
        assert np.max(np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)) < tol


# ----------------------------------------------------------------------------- NEXT-1: full-N pass

def test_regular_all_equals_identity_block_and_energy(oracle):
    """nb_regular_all (P:111 initialisation pass; P:69/P:148 potential energy) = nb_regular with the
    identity block, bit for bit; with h2 = 0 the potentials give W = 1/2 sum m phi, compared with the
    oracle's and with the Plummer closed form -3 pi/32 G M^2 / a within finite-N scatter."""
    cfg = nbgen.make_config(2, N=20000, n_i=64)
    N, cap = cfg["N"], cfg["cap"]
    ctx = open_ctx(cfg)
    ident = np.arange(N, dtype=np.int32)
    a = gpu_regular(ctx, ident, cfg["h2_all"])
    mk = lambda *s, dt=torch.float64: torch.empty(*s, dtype=dt, device="cuda")
    out = dict(acc=mk(N, 3), jerk=mk(N, 3), pot=mk(N), nnb=mk(N, dt=torch.int32),
               nblist=torch.full((N, cap), -1, dtype=torch.int32, device="cuda"), overflow=mk(N, dt=torch.int32))
    ctx.regular_all(_dev(cfg["h2_all"]), **out)
    ctx.synchronize()
    b = parity.to_numpy(out)
    for key in ("acc", "jerk", "pot", "nnb", "overflow"):
        assert np.array_equal(a[key], b[key])
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    sel = np.sort(np.random.default_rng(3).choice(N, 300, replace=False)).astype(np.int32)
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, sel, cfg["h2_all"][sel], cap)
    parity.compare({k: v[sel] for k, v in b.items()}, ref, cap)
    # counts only (nblist = NULL), h2 = 0: full potential of every particle -> potential energy
    out["nnb"].fill_(-1)
    ctx.regular_all(_dev(np.zeros(N)), out["acc"], out["jerk"], out["pot"], out["nnb"], None, out["overflow"])
    ctx.synchronize()
    assert int(out["nnb"].abs().sum()) == 0
    W = 0.5 * float((torch.from_numpy(cfg["m"]).cuda() * out["pot"]).sum())
    tot = oracle.regular(cfg["m"], xp, vp, ident, np.zeros(N), cap, want_list=False)
    W_orc = 0.5 * float((cfg["m"] * tot["pot"]).sum())
    assert abs(W - W_orc) < 1e-6 * abs(W_orc)
    W_plummer = -3.0 * np.pi / 32.0 / cfg["a_plummer"]
    assert abs(W / W_plummer - 1.0) < 0.1        # Kroupa masses: scatter dominated by the few heavy stars


def test_list_rows_sorted_and_bitwise_reproducible(oracle):
    """Rows come back in ascending order (= the oracle's rows, entry by entry, away from band pairs)
    and the whole output is identical run to run."""
    cfg = nbgen.make_config(2, N=30000, n_i=777)
    ctx = open_ctx(cfg)
    a = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    b = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    ref = oracle.regular(cfg["m"], xp, vp, cfg["idx_i"], cfg["h2_i"], cfg["cap"])
    same = 0
    for k in range(777):
        c = min(a["nnb"][k], cfg["cap"])
        assert np.all(np.diff(a["nblist"][k, :c]) > 0)
        if a["nnb"][k] <= cfg["cap"]:
            assert np.array_equal(a["nblist"][k, :c], b["nblist"][k, :c])
            same += int(a["nnb"][k] == ref["nnb"][k] and np.array_equal(a["nblist"][k, :c], ref["nblist"][k, :c]))
    assert same >= 770                                  # all rows but the few holding a flipped band pair
    ctx4 = open_ctx(cfg, cap=4096)                      # long rows: 16 KB of shared memory per warp
    h2 = cfg["h2_i"] * 9.0
    g = gpu_regular(ctx4, cfg["idx_i"], h2)
    assert g["nnb"].max() > 1024
    for k in range(0, 777, 7):
        c = min(g["nnb"][k], 4096)
        assert np.all(np.diff(g["nblist"][k, :c]) > 0)


# ----------------------------------------------------------------------------- NEXT-2 / NEXT-3

def test_irregular_force_matches_oracle_and_completes_the_total(oracle):
    """nb_irregular on the lists nb_regular wrote: FP64 parity with the oracle on the SAME
    lists at the block time and at an intermediate (irregular-step) time, and regular + irregular =
    total direct force within the regular kernel's tolerances."""
    cfg = nbgen.make_config(3, N=40000, n_i=1500)
    ctx = open_ctx(cfg)
    idx, h2 = cfg["idx_i"], cfg["h2_i"]
    reg = ctx.regular_alloc(_dev(idx, torch.int32), _dev(h2))
    n = idx.size
    out = dict(acc=torch.empty((n, 3), dtype=torch.float64, device="cuda"),
               jerk=torch.empty((n, 3), dtype=torch.float64, device="cuda"),
               pot=torch.empty(n, dtype=torch.float64, device="cuda"))
    st = [cfg[k] for k in ("m", "x0", "v0", "a0", "j0", "t0")]
    lst, nnb = reg["nblist"].cpu().numpy(), reg["nnb"].cpu().numpy()
    for t in (cfg["t"], cfg["t"] + 2.0 ** -12):
        ctx.irregular(t, _dev(idx, torch.int32), reg["nnb"], reg["nblist"], **out)
        ctx.synchronize()
        ref = oracle.irregular(*st, t, idx, nnb, lst, cfg["cap"])
        for key, tol in (("acc", 1e-12), ("jerk", 1e-11), ("pot", 1e-12)):
            g = out[key].cpu().numpy().reshape(n, -1); r = ref[key].reshape(n, -1)
            sc = np.linalg.norm(r, axis=1)
            assert np.max(np.linalg.norm(g - r, axis=1) / np.where(sc > 0, sc, 1.0)) < tol, key
    # at the block time: regular (FP32 pair math) + irregular (FP64) = total of the oracle
    ctx.irregular(cfg["t"], _dev(idx, torch.int32), reg["nnb"], reg["nblist"], **out)
    ctx.synchronize()
    xp, vp = oracle.predict(*st[1:], cfg["t"])
    tot = oracle.regular(cfg["m"], xp, vp, idx, np.zeros(n), cfg["cap"], want_list=False)
    assert int(reg["overflow"].sum()) == 0
    for key, tol in (("acc", 1e-5), ("jerk", 1e-4), ("pot", 1e-6)):
        g = (reg[key] + out[key]).cpu().numpy().reshape(n, -1); r = tot[key].reshape(n, -1)
        assert np.max(np.linalg.norm(g - r, axis=1) / np.linalg.norm(r, axis=1)) < tol, key
    # large blocks predict every body once into 64 B records and gather those (NB_TUNE_IRR_PRED_MIN): the same bits
    base = {k: v.clone() for k, v in out.items()}
    ctx.tune("irr_pred_min", 1)
    for v in out.values():
        v.zero_()
    ctx.irregular(cfg["t"], _dev(idx, torch.int32), reg["nnb"], reg["nblist"], **out)
    ctx.synchronize()
    assert all(torch.equal(out[k], base[k]) for k in out)
    ctx.tune("irr_pred_min", 49152)
    # pot = NULL is allowed; an empty list gives exact zeros
    z = torch.zeros(n, dtype=torch.int32, device="cuda")
    ctx.irregular(cfg["t"], _dev(idx, torch.int32), z, reg["nblist"], out["acc"], out["jerk"], None)
    ctx.synchronize()
    assert not out["acc"].any() and not out["jerk"].any()


def test_update_j_equals_full_set_j(oracle):
    """nb_update_j (incremental Send.R): replacing a subset gives bit-identical results to a full
    nb_set_j of the merged state; the predicted records are marked stale."""
    import paper_1504_03687_b200 as nb
    from paper_1504_03687_b200 import NbregError
    cfg = nbgen.make_config(2, N=12000, n_i=300)
    rng = np.random.default_rng(2)
    sub = np.sort(rng.choice(cfg["N"], 999, replace=False)).astype(np.int32)
    new = {k: cfg[k].copy() for k in ("m", "x0", "v0", "a0", "j0", "t0")}
    for k in ("x0", "v0", "a0", "j0"):
        new[k][sub] += rng.normal(size=(999, 3)) * 1e-3
    new["t0"][sub] = cfg["t"] - 2.0 ** -9
    new["m"][sub] *= 1.01
    ctx = open_ctx(cfg)
    ctx.update_j(_dev(sub, torch.int32), *(_dev(new[k][sub]) for k in ("m", "x0", "v0", "a0", "j0", "t0")))
    with pytest.raises(NbregError) as e:
        ctx.regular_alloc(_dev(cfg["idx_i"], torch.int32), _dev(cfg["h2_i"]))
    assert e.value.code == nb.NB_ESTATE
    ctx.predict_all(cfg["t"])
    a = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    cfg2 = dict(cfg); cfg2.update(new)
    ctx2 = open_ctx(cfg2)
    b = gpu_regular(ctx2, cfg["idx_i"], cfg["h2_i"])
    for key in ("acc", "jerk", "pot", "nnb", "overflow"):
        assert np.array_equal(a[key], b[key]), key
    fits = a["nnb"] <= cfg["cap"]
    assert np.array_equal(a["nblist"][fits], b["nblist"][fits])
    check(oracle, ctx, cfg2)


# ----------------------------------------------------------------------------- ADVICE r1 regressions

def test_two_live_contexts_with_different_caps(oracle):
    """The dynamic shared-memory limit of the finalize kernel is per function, not per context: opening a
    second context with a small cap must not break the list sort of an older one with a large cap."""
    cfg = nbgen.make_config(2, N=30000, n_i=300)
    ctx_big = open_ctx(cfg, cap=4096)
    h2 = cfg["h2_i"] * 9.0
    before = gpu_regular(ctx_big, cfg["idx_i"], h2)
    ctx_small = open_ctx(cfg, cap=64)                    # opened later, needs 256 B of sort memory per row
    small = gpu_regular(ctx_small, cfg["idx_i"], cfg["h2_i"])
    after = gpu_regular(ctx_big, cfg["idx_i"], h2)       # the older context, used after the newer was opened
    assert before["nnb"].max() > 1024
    for key in ("acc", "jerk", "pot", "nnb", "overflow"):
        assert np.array_equal(before[key], after[key]), key
    for k in range(300):                                 # sorted rows; an overflowed row keeps ANY cap entries (R10)
        c = before["nnb"][k]
        if c <= 4096:
            assert np.array_equal(before["nblist"][k, :c], after["nblist"][k, :c])
            assert np.all(np.diff(after["nblist"][k, :c]) > 0)
    assert np.isfinite(small["acc"]).all()
    ctx_small.close(); ctx_big.close()


def test_shard_call_checks_time_and_handles_blocks_larger_than_the_shard(oracle):
    """nb_regular_shard: a t other than the predicted one is NB_ESTATE (the body would miss its own record
    at r = 0); a block larger than the shard (n_i > N_shard: the row counters are regrown) works; and
    parallel.regular_jsharded drives a REAL context (world size 1: combine() without collectives) to the
    same result as the unsharded call."""
    import paper_1504_03687_b200 as nb
    from paper_1504_03687_b200 import parallel as par
    cfg = nbgen.make_config(2, N=6000, n_i=16)
    N, cap, t = cfg["N"], cfg["cap"], cfg["t"]
    n_i = 2500
    idx_np = np.sort(np.random.default_rng(5).choice(N, n_i, replace=False)).astype(np.int32)
    h2_np = cfg["h2_all"][idx_np]
    whole = gpu_regular(open_ctx(cfg), idx_np, h2_np)
    idx, h2 = _dev(idx_np, torch.int32), _dev(h2_np)
    b = par.shard_bounds(N, 3)                               # shards of 2048, 2048, 1904 bodies < n_i
    states = [{k: _dev(cfg[k][b[r]:b[r + 1]]) for k in par.STATE_KEYS} for r in range(3)]
    ist = sum(par.gather_istate(states[r], b[r], idx) for r in range(3)).contiguous()
    parts = []
    for r in range(3):
        ctx = nb.nb_open(b[r + 1] - b[r], cap)
        nb.nb_set_j(ctx, *(states[r][k] for k in par.STATE_KEYS))
        ctx.set_j_offset(b[r])
        ctx.predict_all(t)
        part = {k: torch.empty_like(v) for k, v in
                dict(acc=torch.empty((n_i, 3), dtype=torch.float64, device="cuda"),
                     jerk=torch.empty((n_i, 3), dtype=torch.float64, device="cuda"),
                     pot=torch.empty(n_i, dtype=torch.float64, device="cuda"),
                     nnb=torch.empty(n_i, dtype=torch.int32, device="cuda"),
                     nblist=torch.empty((n_i, cap), dtype=torch.int32, device="cuda"),
                     overflow=torch.empty(n_i, dtype=torch.int32, device="cuda")).items()}
        with pytest.raises(nb.NbregError) as e:
            ctx.regular_shard(t + 2.0 ** -20, idx, ist, h2, **part)
        assert e.value.code == nb.NB_ESTATE
        ctx.regular_shard(t, idx, ist, h2, **part)
        ctx.synchronize()
        parts.append(part)
        if r == 1:       # host step on a shard context with an offset is refused (its indices would be local)
            with pytest.raises(nb.NbregError) as e:
                z = np.zeros
                ctx.step_host(*(np.ascontiguousarray(cfg[k][b[1]:b[2]]) for k in par.STATE_KEYS), t,
                              np.zeros(1, np.int32), z(1), z((1, 3)), z((1, 3)), z(1), z(1, np.int32),
                              np.zeros((1, cap), np.int32), z(1, np.int32))
            assert e.value.code == nb.NB_ESTATE
        ctx.close()
    rows = torch.stack([p_["nblist"] for p_ in parts]); cnts = torch.stack([p_["nnb"].long() for p_ in parts])
    nblist, nnb, ovf = par.merge_list_rows(rows, cnts, cap)
    assert np.array_equal(nnb.cpu().numpy(), whole["nnb"])
    for key in ("acc", "jerk", "pot"):
        tot = sum(p_[key] for p_ in parts).cpu().numpy()
        assert np.abs(tot - whole[key]).max() <= 5e-7 * np.abs(whole[key]).max()
    # the production branch of regular_jsharded with a real context, one rank holding everything
    ctx = open_ctx(cfg)
    full_state = {k: _dev(cfg[k]) for k in par.STATE_KEYS}
    got = par.regular_jsharded(ctx, full_state, 0, t, idx, h2)
    ctx.synchronize()
    got = parity.to_numpy(got)
    assert np.array_equal(got["nnb"], whole["nnb"]) and np.array_equal(got["overflow"], whole["overflow"])
    fits = whole["nnb"] <= cap
    mask = np.arange(cap)[None, :] < whole["nnb"][:, None]
    assert np.array_equal(got["nblist"][fits][mask[fits]], whole["nblist"][fits][mask[fits]])
    for key in ("acc", "jerk", "pot"):
        assert np.abs(got[key] - whole[key]).max() <= 5e-7 * np.abs(whole[key]).max()
    ctx.close()


# ----------------------------------------------------------------------------- local frame, fused predictor

def _warp_stats(ctx, fn):
    ctx.tune("stats", 1)
    out = fn()
    loc, tot = ctx.info("local_warps"), ctx.info("total_warps")
    ctx.tune("stats", 0)
    return out, loc, tot


@pytest.mark.parametrize("n_i", [5, 8, 16, 32, 64, 128, 300, 2000])
def test_local_frame_and_hilo_agree_and_match_the_oracle(oracle, n_i):
    """A compact block (config 3: the n_i deepest-level = innermost bodies) takes the warp-local frame (one
    add per component); with the guard switched off (G = 0) the same call differences hi/lo pairs.  Both
    must match the oracle and each other far inside the tolerances, with identical lists outside the band."""
    cfg = nbgen.make_config(3, N=50000, n_i=n_i)
    ctx = open_ctx(cfg)
    ctx.tune("fuse_predict", 0)                       # records on both sides: only the frame differs
    (rep, loc_out, _), loc, tot = _warp_stats(ctx, lambda: check(oracle, ctx, cfg))
    assert tot > 0 and loc == tot, (loc, tot)          # every warp passed the guard
    ctx.tune("local_g_milli", 0)
    (rep0, hl_out, _), loc0, tot0 = _warp_stats(ctx, lambda: check(oracle, ctx, cfg))
    assert loc0 == 0 and tot0 == tot
    print("local frame", n_i, rep, "| hi/lo", rep0)
    assert np.abs(loc_out["nnb"].astype(int) - hl_out["nnb"].astype(int)).max() <= 1      # band pairs only
    same = loc_out["nnb"] == hl_out["nnb"]
    assert same.mean() > 0.98
    for key, tol in (("acc", 3e-6), ("jerk", 3e-5), ("pot", 3e-7)):
        a = loc_out[key].reshape(n_i, -1)[same]; b = hl_out[key].reshape(n_i, -1)[same]
        assert np.max(np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)) < tol, key


def test_scattered_and_two_subcluster_blocks_fall_back_to_hilo(oracle):
    """Adversarial blocks for the local frame: (i) config 2's block of uniformly random indices (a warp's i
    span the whole cluster), (ii) a block made of two far-apart compact groups interleaved so that every
    warp holds members of both, (iii) h2 = 0 (no neighbours: close regular pairs).  The guard must send
    these warps to the hi/lo path, and the results must still meet the tolerances."""
    cfg = nbgen.make_config(2, N=40000, n_i=512)
    ctx = open_ctx(cfg)
    (rep, _, _), loc, tot = _warp_stats(ctx, lambda: check(oracle, ctx, cfg))
    assert loc < tot // 4, (loc, tot)
    r = np.linalg.norm(cfg["x0"], axis=1)
    inner = np.argsort(r)[:128]
    far = np.argsort(np.linalg.norm(cfg["x0"] - np.array([1.5, 0, 0]), axis=1))[:128]
    idx = np.empty(256, np.int32); idx[0::2] = inner; idx[1::2] = far
    assert len(set(idx.tolist())) == 256
    h2 = cfg["h2_all"][idx]
    (rep2, _, _), loc, tot = _warp_stats(ctx, lambda: check(oracle, ctx, cfg, idx_i=idx, h2_i=h2))
    assert loc == 0 and tot > 0
    idx3 = np.sort(inner[:64]).astype(np.int32)
    (rep3, got3, _), loc, tot = _warp_stats(ctx, lambda: check(oracle, ctx, cfg, idx_i=idx3, h2_i=np.zeros(64)))
    assert loc == 0 and got3["nnb"].sum() == 0
    print("fallbacks", rep, rep2, rep3)


@pytest.mark.parametrize("n_i", [1, 5, 8, 13, 16, 31, 32, 64, 100, 128])
def test_fused_predictor_equals_the_two_kernel_route(oracle, n_i):
    """nb_predict_all + nb_regular on a small block predicts inside the force kernel (FP64 state in, no
    records written).  With hi/lo differencing on both routes (G = 0) the records are bit for bit the
    predictor kernel's, so the outputs are IDENTICAL; with the local frame they agree to rounding.  Ragged N."""
    cfg = nbgen.make_config(3, N=9001 if n_i < 100 else 70001, n_i=n_i)
    out = {}
    for g in (0, 4000):
        for fuse in (1, 0):
            ctx = open_ctx(cfg)                      # set_j + predict_all (deferred)
            ctx.tune("fuse_predict", fuse)
            ctx.tune("local_g_milli", g)
            out[g, fuse] = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
            assert ctx.info("last_fused") == fuse
            if fuse:                                 # the pending prediction survives: a larger block still works
                big = nbgen.active_block(cfg, 700)
                gpu_regular(ctx, *big)
                assert ctx.info("last_fused") == 0
                again = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
                assert ctx.info("last_fused") == 0   # the records exist now
                for key in ("nnb", "overflow"):
                    assert np.array_equal(again[key], out[g, fuse][key])
            ctx.close()
    for key in ("acc", "jerk", "pot", "nnb", "overflow"):
        assert np.array_equal(out[0, 1][key], out[0, 0][key]), key
    fits = out[0, 1]["nnb"] <= cfg["cap"]
    assert np.array_equal(out[0, 1]["nblist"][fits], out[0, 0]["nblist"][fits])
    for key, tol in (("acc", 2e-6), ("jerk", 2e-5), ("pot", 2e-7)):
        a = out[4000, 1][key].reshape(n_i, -1); b = out[0, 0][key].reshape(n_i, -1)
        assert np.max(np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)) < tol, key
    ctx = open_ctx(cfg)
    rep, _, _ = check(oracle, ctx, cfg)
    assert ctx.info("last_fused") == 1
    print("fused", n_i, rep)


@pytest.mark.parametrize("k,N,n_i", [(2, 40000, 5000), (3, 70001, 20000)])
def test_morton_reordered_block_equals_callers_order(oracle, k, N, n_i):
    """Blocks of >= 4096 particles are put in Morton order inside the library (a3) so that the 64 particles of
    a warp sit close together and take the local frame.  Outputs must come back in the CALLER's order: same
    counts and lists as the un-reordered call, sums equal to rounding, oracle parity, bitwise reproducible;
    n_i = 5000 sorts in one shared-memory chunk, 20000 (padded to 32768) takes the global merge steps too.
    Config 2's block is scattered over the whole cluster: without the reordering no warp passes the guard."""
    cfg = nbgen.make_config(k, N=N, n_i=n_i)
    if cfg["idx_i"].shape[0] != n_i:
        cfg["idx_i"], cfg["h2_i"] = nbgen.active_block(cfg, n_i)
    ctx = open_ctx(cfg)
    ctx.tune("reorder_min", 0)
    plain, loc0, tot0 = _warp_stats(ctx, lambda: gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"]))
    assert ctx.info("last_reordered") == 0
    ctx.tune("reorder_min", 4096)
    (rep, got, _), loc, tot = _warp_stats(ctx, lambda: check(oracle, ctx, cfg))
    assert ctx.info("last_reordered") == 1
    print("reordered", k, n_i, rep, "local warps", loc, "/", tot, "without reordering", loc0, "/", tot0)
    assert loc > 0.75 * tot and loc >= loc0           # (runs of 64 along the curve that straddle a jump, and halo outliers, fall back)
    assert k != 2 or loc >= 5 * loc0                  # the scattered block: hardly any warp passes without the reordering
    again = gpu_regular(ctx, cfg["idx_i"], cfg["h2_i"])
    for key in ("acc", "jerk", "pot", "nnb", "overflow"):
        assert np.array_equal(got[key], again[key]), key                      # bitwise run to run
    assert np.abs(got["nnb"].astype(int) - plain["nnb"].astype(int)).max() <= 1      # band pairs only
    same = got["nnb"] == plain["nnb"]
    fits = same & (got["nnb"] <= cfg["cap"])
    mask = np.arange(cfg["cap"])[None, :] < got["nnb"][:, None]
    rows_equal = [(np.array_equal(got["nblist"][r][mask[r]], plain["nblist"][r][mask[r]])) for r in np.flatnonzero(fits)]
    assert np.mean(rows_equal) > 0.99
    assert same.mean() > 0.99
    for key, tol in (("acc", 3e-6), ("jerk", 3e-5), ("pot", 3e-7)):       # rows with the same classification of every pair
        a = got[key].reshape(n_i, -1)[same]; b = plain[key].reshape(n_i, -1)[same]
        assert np.max(np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)) < tol, key


def test_regular_all_at_the_papers_size(oracle):
    """SURVEY 8(f) NEXT-1 at the size the paper runs it (initialisation of forces and neighbour lists
    and the O(N^2) potential energy of a million-body run): nb_regular_all at N = 1,048,576 (config 4) with
    lists on a 2 GiB buffer, 1024 seeded rows against the oracle; then counts only (nblist = NULL) with
    h2 = 0: W = 1/2 sum m phi against the Plummer closed form -3 pi / 32 G M^2 / a = -0.3843 (config 4's a)."""
    cfg, ctx, (xp, vp) = _config4(oracle)
    N, cap = cfg["N"], cfg["cap"]
    mk = lambda *s, dt=torch.float64: torch.empty(*s, dtype=dt, device="cuda")
    out = dict(acc=mk(N, 3), jerk=mk(N, 3), pot=mk(N), nnb=mk(N, dt=torch.int32),
               nblist=torch.empty((N, cap), dtype=torch.int32, device="cuda"), overflow=mk(N, dt=torch.int32))
    h2_all = _dev(cfg["h2_all"])
    ctx.regular_all(h2_all, **out)
    ctx.synchronize()
    assert ctx.info("last_reordered") == 1
    sel = np.sort(np.random.default_rng(11).choice(N, 1024, replace=False)).astype(np.int32)
    sel_d = _dev(sel).long()
    got = {k: v[sel_d].cpu().numpy() for k, v in out.items()}
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, sel, cfg["h2_all"][sel], cap)
    rep = parity.compare(got, ref, cap)
    print("regular_all N=1M sample", rep, "S", ctx.info("last_jsplit"))
    nnb_all = out["nnb"].cpu().numpy()
    assert 100 < np.median(nnb_all) < 220          # (halo bodies get radii that hold far more: the median is the target)
    del out["nblist"]
    torch.cuda.empty_cache()
    # potential energy: h2 = 0, counts only
    ctx.regular_all(_dev(np.zeros(N)), out["acc"], out["jerk"], out["pot"], out["nnb"], None, out["overflow"])
    ctx.synchronize()
    assert int(out["nnb"].abs().sum()) == 0
    m_d = _dev(cfg["m"])
    W = 0.5 * float((m_d * out["pot"]).sum())
    f = (m_d[:, None] * out["acc"]).sum(0).cpu().numpy()                       # momentum conservation of the whole pass
    ftot = float((m_d[:, None] * out["acc"]).abs().sum())
    tot = oracle.regular(cfg["m"], xp, vp, sel, np.zeros(1024), cap, want_list=False)
    pg = out["pot"][sel_d].cpu().numpy()
    assert np.max(np.abs(pg - tot["pot"]) / np.abs(tot["pot"])) < 1e-6
    a_pl = cfg["a_plummer"]
    W_plummer = -3.0 * np.pi / 32.0 / a_pl
    # the generator rejects r > 25 a (SURVEY 8(d) recipe), i.e. samples the model truncated there and renormalised
    # to M = 1: W_trunc = -(1 / f^2) int_0^25a G M(r) dM(r) / r, f = M(25 a) -- 0.48 % more bound than the infinite sphere
    r = np.linspace(0.0, 25.0 * a_pl, 2000001)[1:]
    Mr = r**3 / (r * r + a_pl * a_pl) ** 1.5
    rho = 3.0 / (4.0 * np.pi * a_pl**3) * (1.0 + r * r / a_pl**2) ** -2.5
    W_trunc = -np.trapezoid(Mr * rho * 4.0 * np.pi * r, r) / Mr[-1] ** 2
    print("W", W, "Plummer", W_plummer, "truncated at 25a", W_trunc, "ratio", W / W_trunc,
          "|sum m a| / sum |m a|", np.abs(f).max() / ftot)
    assert abs(W_trunc / W_plummer - 1.0046) < 3e-4
    # finite-N scatter with the Kroupa IMF (a few 100-Msun stars carry ~1e-4 of the mass each): ~0.3 % (1 sigma)
    assert abs(W / W_trunc - 1.0) < 0.008
    assert np.abs(f).max() < 1e-6 * ftot
