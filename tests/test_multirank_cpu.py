"""world_size-2 `gloo` test of the N>1 host logic (no GPU): i-sharding of one active block over ranks
(the paper's copy algorithm, P:59 -- every rank holds all j, ranks split the active set, no data-path
collective), max-over-ranks timing reduction, and that the concatenated shard results equal the
unsharded result.  The per-rank compute stands in with the CPU oracle (tests may call it)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import nbgen


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    cfg = nbgen.make_config(3, N=4096, n_i=301)              # ragged: 301 = 150 + 151
    idx, h2 = nbgen.shard_active_block(cfg["idx_i"], cfg["h2_i"], rank, world)
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    out = oracle.regular(cfg["m"], xp, vp, idx, h2, cfg["cap"])
    ms = torch.tensor([10.0 + rank], dtype=torch.float64)    # stand-in per-rank device time
    dist.barrier()
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    pairs = torch.tensor([idx.size * cfg["N"]], dtype=torch.int64)
    dist.all_reduce(pairs, op=dist.ReduceOp.SUM)
    q.put((rank, idx.size, out["acc"], out["nnb"], float(ms.item()), int(pairs.item())))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_i_sharding_gloo(oracle):
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg = nbgen.make_config(3, N=4096, n_i=301)
    full = oracle.regular_step(cfg)
    assert [g[1] for g in got] == [150, 151]
    assert np.array_equal(np.concatenate([g[2] for g in got]), full["acc"])       # bitwise: each i independent
    assert np.array_equal(np.concatenate([g[3] for g in got]), full["nnb"])
    assert all(g[4] == 11.0 for g in got)                                          # max over ranks
    assert all(g[5] == 301 * 4096 for g in got)                                    # whole-job units


# ----------------------------------------------------------------------------- j-sharding (NEXT-4) host logic

def _jshard_worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_1504_03687_b200 import parallel as par
    cfg = nbgen.make_config(3, N=3000, n_i=77)
    N, cap, t = cfg["N"], 64, cfg["t"]                    # cap 64: some rows overflow once the shards are merged
    b = par.shard_bounds(N, world)
    lo, hi = b[rank], b[rank + 1]
    state = {k: torch.from_numpy(np.ascontiguousarray(cfg[k][lo:hi])) for k in par.STATE_KEYS}

    def compute_shard(t_, idx_global, ist, h2):
        """The shard's partial result with the CPU oracle standing in for the library call: local bodies
        plus massless copies of the active bodies other shards own (so that they can be i-particles)."""
        idx = idx_global.numpy().astype(np.int64)
        ist = ist.numpy()
        mine = (idx >= lo) & (idx < hi)
        ext = np.flatnonzero(~mine)
        cat = lambda loc, rows: np.concatenate([loc, ist[rows][:, ext].T])
        m = np.concatenate([cfg["m"][lo:hi], np.zeros(len(ext))])
        x0 = cat(cfg["x0"][lo:hi], [1, 2, 3]); v0 = cat(cfg["v0"][lo:hi], [4, 5, 6])
        a0 = cat(cfg["a0"][lo:hi], [7, 8, 9]); j0 = cat(cfg["j0"][lo:hi], [10, 11, 12])
        t0 = np.concatenate([cfg["t0"][lo:hi], ist[13, ext]])
        where = np.empty(len(idx), np.int32)
        where[mine] = idx[mine] - lo
        where[~mine] = (hi - lo) + np.arange(len(ext))
        xp, vp = oracle.predict(x0, v0, a0, j0, t0, t_)
        out = oracle.regular(m, xp, vp, where, h2.numpy(), 4096)
        nnb = np.zeros(len(idx), np.int32); rows = np.full((len(idx), cap), -1, np.int32)
        for k in range(len(idx)):
            ent = out["nblist"][k, :out["nnb"][k]]
            ent = ent[ent < hi - lo] + lo                  # drop the massless copies, globalise
            nnb[k] = ent.size
            rows[k, :min(ent.size, cap)] = ent[:cap]
        part = dict(acc=torch.from_numpy(out["acc"]), jerk=torch.from_numpy(out["jerk"]), pot=torch.from_numpy(out["pot"]),
                    nnb=torch.from_numpy(nnb), nblist=torch.from_numpy(rows), overflow=torch.from_numpy((nnb > cap).astype(np.int32)))
        return part, cap

    class StubContext:
        """What parallel.py needs of a context, without a GPU: .cap and regular_shard filling the caller's tensors.
        (The product has no hook for this: the test hands in an object with the context's interface.)"""
        def __init__(self):
            self.cap = cap

        def regular_shard(self, t_, idx_global, ist, h2, **out):
            part, _ = compute_shard(t_, idx_global, ist, h2)
            for key, dst in out.items():
                dst.copy_(part[key])

    res = par.regular_jsharded(StubContext(), state, lo, t, torch.from_numpy(cfg["idx_i"].copy()),
                               torch.from_numpy(cfg["h2_i"].copy()))
    q.put((rank, {k: v.numpy() for k, v in res.items()}))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_j_sharding_gloo(oracle):
    """paper_1504_03687_b200.parallel over gloo, world_size 2: the active particles' state published by
    an all-reduce, the partial sums all-reduced, the list rows all-gathered and merged in shard order."""
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_jshard_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg = nbgen.make_config(3, N=3000, n_i=77)
    cap = 64
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    full = oracle.regular(cfg["m"], xp, vp, cfg["idx_i"], cfg["h2_i"], cap)
    assert full["overflow"].any() and not full["overflow"].all()
    for r in range(world):
        g = got[r]
        for key in ("acc", "jerk", "pot"):
            assert np.abs(g[key] - full[key]).max() <= 1e-12 * np.abs(full[key]).max()
        assert np.array_equal(g["nnb"], full["nnb"]) and np.array_equal(g["overflow"], full["overflow"])
        for k in range(77):
            c = min(full["nnb"][k], cap)
            assert np.array_equal(g["nblist"][k, :c], full["nblist"][k, :c])   # ascending: first cap of the true set
            assert np.all(g["nblist"][k, c:] == -1)
    assert all(np.array_equal(got[0][key], got[1][key]) for key in got[0])      # every rank holds the same result
