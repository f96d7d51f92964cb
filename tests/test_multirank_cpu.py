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
