"""Host-side sharding of the path over ranks (one process per GPU).  No arithmetic of the method lives here.

The path shards by q: "no inter-image communication is required during the outer loop" (the paper's
image level; L229 "embarrassingly parallel over q").  Operators are replicated, every rank runs the single-GPU path on
its own q-points, outputs are disjoint, so there is NO data-path collective; `torch.distributed` is used only for the
barrier, the max-over-ranks of the device time and, if the caller wants one table, a final all-gather of omega_q.

When g(Re,Rp) does not fit one GPU the paper splits Rp over ranks instead (its pool level);
`rp_ranges` gives that split (contiguous Rp slabs, the unit of `epw_interp_set_g_slabs`).
"""
from __future__ import annotations

import numpy as np


def q_ranges(nq: int, world: int) -> list[tuple[int, int]]:
    """Contiguous, disjoint, exhaustive [start, stop) of the q-list for each rank; sizes differ by at most one."""
    if nq < 0 or world <= 0:
        raise ValueError("q_ranges: nq must be >= 0 and world > 0")
    base, extra = divmod(nq, world)
    out, start = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((start, start + n))
        start += n
    return out


def q_block(step: int, world: int, rank: int, nq_step: int, nq: int) -> np.ndarray:
    """Indices of the `nq_step` q-points rank `rank` interpolates in step `step` of a run that walks the q-list in
    blocks of world*nq_step (bench.py): the blocks of the ranks of one step are consecutive and disjoint; the walk
    wraps around the list (weak scaling: every rank always has nq_step q-points)."""
    if not (0 <= rank < world) or nq_step <= 0 or nq <= 0:
        raise ValueError("q_block: bad rank / nq_step / nq")
    start = ((step * world + rank) * nq_step) % nq
    return (start + np.arange(nq_step)) % nq


def rp_ranges(np_: int, world: int) -> list[tuple[int, int]]:
    """Contiguous Rp-slab range [start, stop) per rank for an Rp-split g(Re,Rp)."""
    return q_ranges(np_, world)


def max_over_ranks_ms(ms: float, dist=None, device=None) -> float:
    """Device time of a step = max over ranks (a collective on one double; identity without a process group)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch

    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def all_gather_rows(local, ranges, dist, device=None):
    """Gather per-rank row blocks (e.g. omega_q [nq_local][Nm]) into the full table on every rank.  Blocks may differ
    in size by one row (q_ranges); they are padded to the largest for the collective."""
    import torch

    world = dist.get_world_size()
    nmax = max(b - a for a, b in ranges)
    pad = torch.zeros((nmax,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad)
    return torch.cat([parts[r][: ranges[r][1] - ranges[r][0]] for r in range(world)], dim=0)


def interpolate_rp_sharded(epw, handle, q_list, nq, rows, run_rest, dist=None, reduce_fn=None):
    """One interpolation step with g(Re,Rp) split by Rp over the ranks: every rank contracts its own
    slabs (`epw_interp_rp_to_q_partial`), the partial g(Re,q) are summed across ranks ON THE DEVICE and on the current
    stream (NCCL all-reduce through torch.distributed -- the paper stages this through the host, L514-522), then
    `run_rest()` (the caller's `epw_interp_interpolate[_grid]` on this rank's share of the k-points) runs with S1
    replaced by the reduced g(Re,q).  `reduce_fn(tensor)` overrides the collective (tests on one GPU sum explicitly).
    Returns the reduced g(Re,q) tensor [nq][rows][2] (kept alive by the caller until the stream has completed)."""
    import torch

    g1 = torch.empty((nq, rows, 2), dtype=torch.float64, device=q_list.device)
    epw.epw_interp_rp_to_q_partial(handle, q_list, nq, g1)
    if reduce_fn is not None:
        g1 = reduce_fn(g1)
    elif dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(g1, op=dist.ReduceOp.SUM)
    epw.epw_interp_set_gq(handle, g1)
    try:
        run_rest()
    finally:
        epw.epw_interp_set_gq(handle, None)
    return g1


def k_ranges(nk: int, world: int) -> list[tuple[int, int]]:
    """After the all-reduce every rank holds g(Re,q) and interpolates its own contiguous share of the k-list."""
    return q_ranges(nk, world)
