"""j-sharded regular force over the ranks of a torch.distributed group.

P:127: "each GPU has a similar particle dataset size ... all GPUs in the same node together access the
complete particle dataset"; Table 2: calculation O(N_i N) against communication O(N_i).  Every
rank owns a contiguous shard of the bodies in its own `NbContext` (nb_open(N_shard), nb_set_j,
nb_set_j_offset) and evaluates its shard's contribution to the active block with nb_regular_shard;
what crosses the wire per active particle is its 14-double state (in, one all-reduce with a single non-zero
contributor per column: exact), 7 doubles + 1 count per shard (all-gather, summed in rank order: deterministic)
and its list row (all-gather).  The collectives are plain `torch.distributed` calls
(NCCL over NVLink on GPUs, gloo in the CPU tests): a few hundred KB against milliseconds of pair
arithmetic -- there is no compute step to fuse them into.

Marshalling and collectives only: every pair interaction runs in the library's kernels.
"""
from __future__ import annotations

import torch
import torch.distributed as dist

STATE_KEYS = ("m", "x0", "v0", "a0", "j0", "t0")       # order of nb_set_j and of the istate rows


def _world(group=None) -> int:
    return dist.get_world_size(group) if dist.is_initialized() else 1


def _via_host(t: torch.Tensor, group=None) -> bool:
    """gloo has no CUDA all_gather: with that backend (two ranks sharing one GPU in the tests) the few hundred
    KB of a block go through host memory; NCCL takes the device tensors as they are."""
    return t.is_cuda and dist.get_backend(group) == "gloo"


def _all_reduce_sum(t: torch.Tensor, group=None) -> torch.Tensor:
    if _world(group) == 1:
        return t
    if _via_host(t, group):
        h = t.cpu()
        dist.all_reduce(h, op=dist.ReduceOp.SUM, group=group)
        return h.to(t.device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t


def _all_gather(t: torch.Tensor, group=None) -> torch.Tensor:
    """[world, *t.shape], rank order."""
    world = _world(group)
    if world == 1:
        return t[None]
    src = t.cpu().contiguous() if _via_host(t, group) else t.contiguous()
    parts = [torch.empty_like(src) for _ in range(world)]
    dist.all_gather(parts, src, group=group)
    return torch.stack(parts).to(t.device)


def shard_bounds(N: int, world: int, tile: int = 256) -> list[int]:
    """Offsets [0 = b_0 <= b_1 <= ... <= b_world = N] of contiguous shards of whole j-tiles (the last
    shard takes the ragged tail), sizes as equal as whole tiles allow."""
    ntiles = -(-N // tile)
    out = [min(N, (ntiles * r // world) * tile) for r in range(world)]
    return out + [N]


def gather_istate(state: dict, offset: int, idx_global: torch.Tensor, group=None) -> torch.Tensor:
    """istate[14][n_i] of the active particles (global indices idx_global) from the shards that own
    them: each rank fills the columns of its own bodies, the rest stay zero, one all-reduce (SUM) --
    exact, since every column has exactly one non-zero contribution."""
    n = idx_global.numel()
    n_loc = state["m"].shape[0]
    loc = idx_global.long() - offset
    mine = (loc >= 0) & (loc < n_loc)
    sel = loc[mine]
    ist = torch.zeros((14, n), dtype=torch.float64, device=idx_global.device)
    ist[0, mine] = state["m"][sel]
    ist[13, mine] = state["t0"][sel]
    for r0, key in ((1, "x0"), (4, "v0"), (7, "a0"), (10, "j0")):
        ist[r0:r0 + 3, mine] = state[key][sel].T
    return _all_reduce_sum(ist, group)


def merge_list_rows(rows: torch.Tensor, counts: torch.Tensor, cap: int):
    """rows[G][n][cap], counts[G][n] (shard order = ascending j) -> (nblist[n][cap], nnb[n], overflow[n]):
    the stored entries of every shard concatenated in shard order, cut at cap; nnb is the true total."""
    G, n, _ = rows.shape
    stored = counts.clamp(max=cap)                                   # entries each shard actually holds
    start = torch.cumsum(stored, dim=0) - stored                     # [G][n] first output column of shard g
    col = torch.arange(cap, device=rows.device)
    dest = start[:, :, None] + col[None, None, :]                    # [G][n][cap]
    valid = (col[None, None, :] < stored[:, :, None]) & (dest < cap)
    out = torch.full((n, cap), -1, dtype=rows.dtype, device=rows.device)
    row_id = torch.arange(n, device=rows.device)[None, :, None].expand(G, n, cap)
    out[row_id[valid], dest[valid]] = rows[valid]
    nnb = counts.sum(dim=0).to(torch.int32)
    return out, nnb, (nnb > cap).to(torch.int32)


def combine(part: dict, cap: int, group=None) -> dict:
    """Per-shard partial outputs of nb_regular_shard -> the block's results on every rank.  The seven sums
    per active particle are all-gathered and added IN RANK ORDER on every rank (not all-reduced: the order of
    an all-reduce is the collective library's choice), so the FP64 result is bitwise the same on every rank
    and from run to run (reading R19; copies must not diverge)."""
    sums = torch.cat([part["acc"], part["jerk"], part["pot"][:, None]], dim=1).contiguous()    # [n][7]
    all_sums = _all_gather(sums, group)                                                         # [G][n][7]
    total = all_sums[0].clone()
    for g in range(1, all_sums.shape[0]):
        total += all_sums[g]
    rows = _all_gather(part["nblist"], group)
    cnts = _all_gather(part["nnb"].to(torch.int64), group)
    nblist, nnb, overflow = merge_list_rows(rows, cnts, cap)
    return dict(acc=total[:, 0:3].contiguous(), jerk=total[:, 3:6].contiguous(), pot=total[:, 6].contiguous(),
                nnb=nnb, nblist=nblist, overflow=overflow)


def regular_jsharded(ctx, state: dict, offset: int, t: float, idx_global: torch.Tensor, h2_i: torch.Tensor,
                     group=None) -> dict:
    """One regular-force block over a j-sharded system.  `ctx` holds this rank's shard (already
    nb_set_j / nb_set_j_offset / nb_predict_all(t)); `state` is the shard's FP64 state (tensors keyed by
    STATE_KEYS) used to publish the active particles' own state.  Returns the full outputs on every
    rank.  The shard's partial sums come from ctx.regular_shard (the library) and from nowhere else."""
    n, cap = idx_global.numel(), ctx.cap
    ist = gather_istate(state, offset, idx_global, group)
    dev, f8, i4 = idx_global.device, torch.float64, torch.int32
    part = dict(acc=torch.empty((n, 3), dtype=f8, device=dev), jerk=torch.empty((n, 3), dtype=f8, device=dev),
                pot=torch.empty(n, dtype=f8, device=dev), nnb=torch.empty(n, dtype=i4, device=dev),
                nblist=torch.full((n, cap), -1, dtype=i4, device=dev), overflow=torch.empty(n, dtype=i4, device=dev))
    ctx.regular_shard(t, idx_global, ist.contiguous(), h2_i, **part)
    return combine(part, cap, group)
