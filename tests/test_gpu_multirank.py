"""SURVEY 8(f) NEXT-4 as an executable multi-rank program: two PROCESSES share the one B200, each opens its own
NbContext over half of the bodies (nb_open(N_shard), nb_set_j, nb_set_j_offset, nb_predict_all) and they run
paper_1504_03687_b200.parallel.regular_jsharded over a gloo process group (NCCL refuses two ranks on one
device) -- the library call, no stand-in.  Every rank must hold the unsharded result = the oracle's."""
import os
import socket

import numpy as np
import pytest

import nbgen
from tests import parity

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_i, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    import paper_1504_03687_b200 as nb
    from paper_1504_03687_b200 import parallel as par
    cfg = nbgen.make_config(2, N=30011, n_i=n_i)
    N, cap, t = cfg["N"], cfg["cap"], cfg["t"]
    b = par.shard_bounds(N, world)
    lo, hi = b[rank], b[rank + 1]
    dev = lambda a, dt=None: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    state = {k: dev(cfg[k][lo:hi]) for k in par.STATE_KEYS}
    ctx = nb.nb_open(hi - lo, cap)
    nb.nb_set_j(ctx, *(state[k] for k in par.STATE_KEYS))
    ctx.set_j_offset(lo)
    ctx.predict_all(t)
    idx, h2 = dev(cfg["idx_i"]), dev(cfg["h2_i"])
    res = par.regular_jsharded(ctx, state, lo, t, idx, h2)
    res2 = par.regular_jsharded(ctx, state, lo, t, idx, h2)          # bitwise reproducible across calls
    ctx.synchronize()
    same = all(torch.equal(res[k], res2[k]) for k in ("acc", "jerk", "pot", "nnb", "overflow"))
    q.put((rank, {k: v.cpu().numpy() for k, v in res.items()}, same, ctx.info("last_reordered")))
    dist.barrier()
    ctx.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("n_i", [333, 5000])
def test_two_processes_on_one_gpu_j_sharded(oracle, n_i):
    import torch.multiprocessing as mp
    world = 2
    mpc = mp.get_context("spawn")
    q = mpc.Queue()
    port = _free_port()
    procs = [mpc.Process(target=_worker, args=(r, world, port, n_i, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = {}
    for _ in range(world):
        r, res, same, reordered = q.get(timeout=600)
        got[r] = res
        assert same
        assert reordered == (1 if n_i >= 4096 else 0)          # the large block took the Morton order inside each shard
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    cfg = nbgen.make_config(2, N=30011, n_i=n_i)
    cap = cfg["cap"]
    xp, vp = oracle.predict(cfg["x0"], cfg["v0"], cfg["a0"], cfg["j0"], cfg["t0"], cfg["t"])
    ref = parity.oracle_reference(oracle, cfg["m"], xp, vp, cfg["idx_i"], cfg["h2_i"], cap)
    rep = parity.compare(got[0], ref, cap)
    print("two processes, j-sharded", n_i, rep)
    for key in got[0]:
        if key == "nblist":
            fits = got[0]["nnb"] <= cap
            assert np.array_equal(got[0][key][fits], got[1][key][fits])
        else:
            assert np.array_equal(got[0][key], got[1][key]), key          # every rank holds the same bits
    # the same block on ONE context holding everything
    import paper_1504_03687_b200 as nb
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ctx = nb.nb_open(cfg["N"], cap)
    nb.nb_set_j(ctx, *(dev(cfg[k]) for k in ("m", "x0", "v0", "a0", "j0", "t0")))
    ctx.predict_all(cfg["t"])
    whole = parity.to_numpy(ctx.regular_alloc(dev(cfg["idx_i"]), dev(cfg["h2_i"])))
    assert np.abs(got[0]["nnb"].astype(int) - whole["nnb"].astype(int)).max() <= 1
    same = got[0]["nnb"] == whole["nnb"]
    for key, tol in (("acc", 3e-6), ("jerk", 3e-5), ("pot", 3e-7)):
        a = got[0][key].reshape(n_i, -1)[same]; b_ = whole[key].reshape(n_i, -1)[same]
        assert np.max(np.linalg.norm(a - b_, axis=1) / np.linalg.norm(b_, axis=1)) < tol, key
    ctx.close()
