"""nb_next_block_static: block selection for callers that cannot allocate GPU memory.

Some users of this library run where a cudaMalloc is off the table: a module loaded into an application whose memory
pool has already taken the whole device, or a hook that runs beside the application's own streams and must not cause
the device-wide synchronisation an allocation brings.  They cannot open a context (nb_open allocates the j-state),
so the ordinary selection call nb_next_block is out of reach.  nb_next_block_static takes t0, dt and the output
buffers from the caller and keeps its few KB of working memory in a fixed array inside the library; the price is a
size limit (NB_STATIC_MAX_N bodies) and that overlapping calls share -- and would race on -- that array.

What is checked here: on the same seeded cluster the new entry point returns exactly what the existing path
(nb_set_j + nb_set_steps + nb_next_block) returns -- block time bit for bit, the same count, the same ascending index
list (integer work: no tolerance) -- on two calls in a row.  The second call's block lies LATER in time than the
first one's, so a minimum left behind in the shared array by the first call would be caught.  The file name sorts
last on purpose: it runs after every other test (the array then holds whatever they left) and, run alone, on a
process in which nothing of the library has executed yet (the first call does the one-time address look-up).
"""
import numpy as np
import pytest

import nbgen

torch = pytest.importorskip("torch")


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _existing_path(cfg, t0, dt):
    """The path the library already had: a context holding the state, nb_set_steps, nb_next_block."""
    import paper_1504_03687_b200 as nb
    N = cfg["N"]
    ctx = nb.nb_open(N, 8)
    nb.nb_set_j(ctx, *(_dev(cfg[k]) for k in ("m", "x0", "v0", "a0", "j0")), _dev(t0))
    ctx.set_steps(_dev(dt))
    idx = torch.full((N,), -1, dtype=torch.int32, device="cuda")
    t_next, n = ctx.next_block(idx)
    out = idx.cpu().numpy()
    ctx.close()
    return t_next, n, out


@pytest.mark.gpu
def test_static_scratch_selection_equals_the_context_path_twice_in_a_row():
    import paper_1504_03687_b200 as nb
    cfg = nbgen.make_config(2, N=70001, n_i=16)              # 35 chunks of 2048 bodies, the last one ragged
    N = cfg["N"]
    dt = 2.0 ** -cfg["levels"].astype(np.float64)
    cases = [(np.floor(0.3 / dt) * dt, dt),                  # first call: the block at t = 0.30005, 30150 bodies
             (np.floor(0.7 / dt) * dt, dt)]                  # second call: a LATER block (t = 0.70001), 9869 bodies
    d_idx = torch.empty(N, dtype=torch.int32, device="cuda")
    d_block = torch.empty(2, dtype=torch.float64, device="cuda")
    got = []
    for t0, step in cases:                                   # the two static calls back to back, nothing in between
        d_idx.fill_(-1)
        nb.nb_next_block_static(_dev(t0), _dev(step), d_idx, d_block)
        torch.cuda.synchronize()
        got.append((d_block.cpu().numpy().copy(), d_idx.cpu().numpy().copy()))
    times = []
    for (t0, step), (block, idx) in zip(cases, got):
        t_ref, n_ref, idx_ref = _existing_path(cfg, t0, step)
        assert block[0] == t_ref and int(block[1]) == n_ref and block[1] == float(n_ref)
        assert 0 < n_ref < N
        assert np.array_equal(idx[:n_ref], idx_ref[:n_ref])          # same bodies, same (ascending) order
        assert np.all(np.diff(idx[:n_ref]) > 0)
        assert np.all(idx[n_ref:] == -1)                             # nothing written past the block
        due = np.flatnonzero(t0 + step == (t0 + step).min())         # and both equal the definition
        assert np.array_equal(idx[:n_ref], due) and t_ref == (t0 + step).min()
        times.append(t_ref)
    assert times[1] > times[0]                                       # a stale minimum would have shown


@pytest.mark.gpu
def test_static_scratch_selection_on_a_side_stream_and_single_body():
    import paper_1504_03687_b200 as nb
    side = torch.cuda.Stream()
    t0 = torch.tensor([0.25], dtype=torch.float64, device="cuda")
    dt = torch.tensor([0.125], dtype=torch.float64, device="cuda")
    idx = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    block = torch.zeros(2, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    nb.nb_next_block_static(t0, dt, idx, block, stream=side)
    side.synchronize()
    assert block.tolist() == [0.375, 1.0] and idx.tolist() == [0]


def test_static_scratch_selection_rejects_sizes_beyond_its_limit_before_touching_the_gpu():
    """Runs without a GPU too: the size and pointer checks come before the first CUDA call."""
    import ctypes
    import paper_1504_03687_b200 as nb
    lib = nb.load_library()
    fake = ctypes.c_void_p(256)                                      # never dereferenced
    assert lib.nb_next_block_static(nb.NB_STATIC_MAX_N + 1, fake, fake, fake, fake, None) == nb.NB_ELIMIT
    assert lib.nb_next_block_static(0, fake, fake, fake, fake, None) == nb.NB_EINVAL
    assert lib.nb_next_block_static(8, None, fake, fake, fake, None) == nb.NB_EINVAL
    assert b"NB_STATIC_MAX_N" in lib.nb_strerror(nb.NB_ELIMIT)
