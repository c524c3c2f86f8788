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


def ghost_planes(lo: int, hi: int, R: int, K: int) -> List[int]:
    """The planes a rank owning [lo, hi) holds as ghosts: the left and right neighbours' planes in the
    order of ghost_sources, each plane once, never one of its own (short periodic boxes alias them)."""
    need_l, need_r = ghost_sources(lo, hi, R, K)
    return [p for p in dict.fromkeys(need_l + need_r) if not lo <= p < hi]


def _owner(plane: int, ranges: Sequence[Tuple[int, int]]) -> int:
    for r, (lo, hi) in enumerate(ranges):
        if lo <= plane < hi:
            return r
    raise ValueError(f"plane {plane} has no owner")


def exchange_ghosts(my_planes: List[torch.Tensor], ranges: Sequence[Tuple[int, int]], R: int, K: int, dist,
                    rank: Optional[int] = None, alloc=None, via_host: bool = False
                    ) -> Tuple[List[torch.Tensor], List[torch.Tensor]]:
    """The one exchange step.  `my_planes[i]` is the float32 [n, 3] array of plane ranges[rank][0] + i.
    Returns (left ghosts, right ghosts), each a list of R arrays in increasing plane order.
    Counts travel first (one int64 per plane), then the positions, as batched isend/irecv pairs, so that
    any mix of neighbours (including a rank that is its own neighbour when world == 1, or a neighbour
    two ranks away when ranges are shorter than R) is served.

    Matching does NOT rely on message tags (NCCL ignores them): for every ordered pair of ranks the sender
    and the receiver enumerate the planes in the same order -- the receiver's need list (left ghosts, then
    right ghosts, increasing slot) -- and the operations of one pair are issued in that order on both sides.
    Empty planes send their count only.  `alloc(slot, n)` may supply the receive buffer of ghost slot
    `slot` (e.g. a slice at the tail of the rank's particle array); `via_host` stages CUDA tensors through
    host memory (for the gloo backend on a GPU box)."""
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
    # per-pair order: sends to `dst` follow dst's slot order (the loop above enumerates them so); receives
    # from `src` follow my own slot order.  Both are "the receiver's need list in increasing slot".
    remote_send.sort(key=lambda t: (t[0], t[1]))
    remote_recv.sort(key=lambda t: (t[0], t[1]))
    xdev = torch.device("cpu") if via_host else dev
    # 1) counts
    ops, cnt_bufs = [], {}
    for dst, slot, pl in remote_send:
        t = torch.tensor([my_planes[pl - lo].shape[0]], dtype=torch.int64, device=xdev)
        ops.append(dist.P2POp(dist.isend, t, dst))
    for src, slot in remote_recv:
        cnt_bufs[slot] = torch.zeros(1, dtype=torch.int64, device=xdev)
        ops.append(dist.P2POp(dist.irecv, cnt_bufs[slot], src))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    # 2) positions (nothing travels for an empty plane: both sides know its count)
    ops, staged = [], []
    for dst, slot, pl in remote_send:
        t = my_planes[pl - lo]
        if t.shape[0] == 0:
            continue
        t = t.contiguous()
        ops.append(dist.P2POp(dist.isend, t.cpu() if via_host else t, dst))
    for src, slot in remote_recv:
        n = int(cnt_bufs[slot].item())
        out[slot] = alloc(slot, n) if alloc is not None else torch.empty(n, 3, dtype=torch.float32, device=dev)
        assert out[slot].shape == (n, 3) and out[slot].is_contiguous()
        if n == 0:
            continue
        if via_host:
            h = torch.empty(n, 3, dtype=torch.float32)
            staged.append((out[slot], h))
            ops.append(dist.P2POp(dist.irecv, h, src))
        else:
            ops.append(dist.P2POp(dist.irecv, out[slot], src))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()
    for dst_t, h in staged:
        dst_t.copy_(h)
    if alloc is not None:                       # ghosts that are my own planes (periodic wrap onto myself) are copied in
        for slot, pl in enumerate(needs):
            if _owner(pl, ranges) == rank:
                buf = alloc(slot, my_planes[pl - lo].shape[0])
                buf.copy_(my_planes[pl - lo])
                out[slot] = buf
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
