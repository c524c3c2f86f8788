"""Host-side plumbing for more than one GPU.

The near-field force shards by contiguous ranges of x-planes of cells (the paper's slab
decomposition): a rank owns the sinks of its planes and needs, as sources
only, the R planes on either side from its x-neighbours.  That is ONE exchange step of
positions (neighbour send/recv, no all-reduce, no output exchange); each rank then calls
nf_stream_slabs (or nf_forces on a resident chunk) on its planes + ghosts.

This module holds no arithmetic of the method: it plans the ranges, moves plane arrays
between ranks with torch.distributed point-to-point calls (gloo on CPU, NCCL on GPUs) and
reduces the numbers bench.py reports.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import torch


def plan_x_slabs(plane_work: Sequence[int], world: int) -> List[Tuple[int, int]]:
    """Cut K planes into `world` contiguous ranges [lo, hi) of near-equal WORK (pairwise
    interactions per plane, not plane counts: clustered boxes are uneven).
    Boundaries are placed where the running sum crosses k/world of the total; every rank gets
    at least one plane when K >= world."""
    K = len(plane_work)
    if world < 1 or K < world:
        raise ValueError("need 1 <= world <= number of planes")
    total = float(sum(plane_work))
    bounds = [0]
    run = 0.0
    k = 1
    for i, wk in enumerate(plane_work):
        run += float(wk)
        # close range k-1 after plane i if the target is reached, keeping enough planes for the rest
        while k < world and (run >= total * k / world or K - (i + 1) == world - k) and i + 1 > bounds[-1]:
            bounds.append(i + 1)
            k += 1
    while len(bounds) < world:                      # degenerate (all-zero work): pad one plane each
        bounds.append(bounds[-1] + 1)
    bounds.append(K)
    return [(bounds[r], bounds[r + 1]) for r in range(world)]


def ghost_sources(lo: int, hi: int, R: int, K: int) -> Tuple[List[int], List[int]]:
    """Plane indices (mod K) a rank owning [lo, hi) needs from the left and from the right."""
    return [(lo - R + j) % K for j in range(R)], [(hi + j) % K for j in range(R)]


def _owner(plane: int, ranges: Sequence[Tuple[int, int]]) -> int:
    for r, (lo, hi) in enumerate(ranges):
        if lo <= plane < hi:
            return r
    raise ValueError(f"plane {plane} has no owner")


def exchange_ghosts(my_planes: List[torch.Tensor], ranges: Sequence[Tuple[int, int]], R: int, K: int, dist,
                    rank: Optional[int] = None) -> Tuple[List[torch.Tensor], List[torch.Tensor]]:
    """The one exchange step.  `my_planes[i]` is the float32 [n, 3] array of plane ranges[rank][0] + i.
    Returns (left ghosts, right ghosts), each a list of R arrays in increasing plane order.
    Counts travel first (one int64 per plane), then the positions, all as isend/irecv pairs
    keyed by the plane index so that any mix of neighbours (including a rank that is its own
    neighbour when world == 1, or a neighbour two ranks away when ranges are shorter than R)
    is served."""
    rank = dist.get_rank() if rank is None else rank
    world = len(ranges)
    lo, hi = ranges[rank]
    dev = my_planes[0].device if my_planes else torch.device("cpu")
    need_l, need_r = ghost_sources(lo, hi, R, K)
    needs = need_l + need_r
    # what the others need from me
    sends = []                                       # (dst rank, slot in dst's need list, plane)
    for dst in range(world):
        dl, dh = ranges[dst]
        nl, nr = ghost_sources(dl, dh, R, K)
        for slot, pl in enumerate(nl + nr):
            if lo <= pl < hi:
                sends.append((dst, slot, pl))
    out: List[Optional[torch.Tensor]] = [None] * len(needs)
    # local copies first (periodic wrap onto oneself)
    remote_recv = []
    for slot, pl in enumerate(needs):
        src = _owner(pl, ranges)
        if src == rank:
            out[slot] = my_planes[pl - lo]
        else:
            remote_recv.append((src, slot))
    remote_send = [(dst, slot, pl) for dst, slot, pl in sends if dst != rank]
    # 1) counts
    ops, cnt_bufs = [], {}
    for dst, slot, pl in remote_send:
        t = torch.tensor([my_planes[pl - lo].shape[0]], dtype=torch.int64, device=dev)
        ops.append(dist.P2POp(dist.isend, t, dst, tag=slot))
    for src, slot in remote_recv:
        cnt_bufs[slot] = torch.zeros(1, dtype=torch.int64, device=dev)
        ops.append(dist.P2POp(dist.irecv, cnt_bufs[slot], src, tag=slot))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    # 2) positions
    ops = []
    for dst, slot, pl in remote_send:
        ops.append(dist.P2POp(dist.isend, my_planes[pl - lo].contiguous(), dst, tag=100 + slot))
    for src, slot in remote_recv:
        out[slot] = torch.empty(int(cnt_bufs[slot].item()), 3, dtype=torch.float32, device=dev)
        ops.append(dist.P2POp(dist.irecv, out[slot], src, tag=100 + slot))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    return out[:R], out[R:]


def reduce_report(step_seconds: float, interactions: int, particles: int, dist=None, device=None):
    """Whole-job numbers for bench.py: time = MAX over ranks, work = SUM over ranks."""
    t = torch.tensor([step_seconds], dtype=torch.float64, device=device)
    wk = torch.tensor([float(interactions), float(particles)], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(wk)
    sec = float(t.item())
    return {"seconds": sec, "interactions": float(wk[0].item()), "particles": float(wk[1].item()),
            "interactions_per_s": float(wk[0].item()) / sec, "particles_per_s": float(wk[1].item()) / sec}
