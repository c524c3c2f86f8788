"""The N > 1 path on CPU: world_size-2 `gloo` run of the slab sharding plumbing
(paper_1810_02916_b200/shard.py): plan by work, ONE neighbour exchange of ghost planes, and
the max/sum reduction bench.py reports.  Each rank then evaluates its own sinks with the
oracle on (ghosts + own planes) and must reproduce the single-process result."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_1810_02916_b200 import inputs, shard

K, R, N = 9, 2, 6000


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _input():
    cfg = inputs.scaled(inputs.config(3), N, K)
    cfg = inputs.dataclasses.replace(cfg, n_halos=6)
    return cfg, inputs.make_positions(cfg).numpy()


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg, pos = _input()
        keys, _ = oracle.keys(pos, K, cfg.box)
        cx = keys // (K * K)
        cnt = np.bincount(keys, minlength=K ** 3).astype(np.uint32)
        work = [oracle.interactions(cnt, K, R, p, p + 1) for p in range(K)]
        ranges = shard.plan_x_slabs(work, world)
        lo, hi = ranges[rank]
        plane_idx = [np.nonzero(cx == p)[0] for p in range(K)]
        mine = [torch.from_numpy(pos[plane_idx[p]]) for p in range(lo, hi)]
        left, right = shard.exchange_ghosts(mine, ranges, R, K, dist)
        need_l, need_r = shard.ghost_sources(lo, hi, R, K)
        for got, pl in zip(left + right, need_l + need_r):            # the exchange delivered the right planes
            assert np.array_equal(got.numpy(), pos[plane_idx[pl]])
        # the same exchange straight into the tail of the rank's particle array (what bench.py's sharded step
        # does): one slot per distinct ghost plane behind the own particles
        ghosts = shard.ghost_planes(lo, hi, R, K)
        n_own = sum(t.shape[0] for t in mine)
        goff, o = {}, n_own
        for pl in ghosts:
            goff[pl] = o
            o += plane_idx[pl].size
        buf = torch.zeros(o, 3)
        buf[:n_own] = torch.cat(mine)
        slot_plane = need_l + need_r
        scratch = {}

        def alloc(slot, n):
            pl = slot_plane[slot]
            if pl in goff:
                return buf[goff[pl]:goff[pl] + n]
            scratch[slot] = torch.empty(n, 3)            # a ghost that is one of my own planes (short periodic box)
            return scratch[slot]
        shard.exchange_ghosts(mine, ranges, R, K, dist, alloc=alloc)
        for pl in ghosts:
            assert np.array_equal(buf[goff[pl]:goff[pl] + plane_idx[pl].size].numpy(), pos[plane_idx[pl]])
        # a plane can be both an own plane and a ghost (short periodic box): use each plane once
        have = {}
        for pl, t in zip(need_l, left):
            have[pl] = t
        for pl, t in zip(need_r, right):
            have[pl] = t
        for p, t in zip(range(lo, hi), mine):
            have[p] = t
        order = sorted(have)
        local = torch.cat([have[p] for p in order]).numpy()
        starts = np.cumsum([0] + [have[p].shape[0] for p in order])
        sink_idx = np.concatenate([np.arange(starts[order.index(p)], starts[order.index(p) + 1]) for p in range(lo, hi)])
        a = oracle.forces(local, K, R, cfg.eps, cfg.box, cfg.Gm, sink_idx=sink_idx)
        orig = np.concatenate([plane_idx[p] for p in range(lo, hi)])
        rep = shard.reduce_report(1.0 + rank, int(sum(work[lo:hi])), int(orig.size), dist)
        q.put((rank, ranges, orig, a, rep))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_slab_sharding_matches_single_process():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = [q.get(timeout=240) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg, pos = _input()
    ref = oracle.forces(pos, K, R, cfg.eps, cfg.box, cfg.Gm)
    seen = np.zeros(N, bool)
    total_I = oracle.interactions(np.bincount(oracle.keys(pos, K, cfg.box)[0], minlength=K ** 3).astype(np.uint32), K, R)
    for rank, ranges, orig, a, rep in results:
        assert not seen[orig].any()
        seen[orig] = True
        scale = np.abs(ref).max()
        assert np.allclose(a, ref[orig], rtol=1e-9, atol=1e-12 * scale)
        assert rep["seconds"] == 2.0 and rep["interactions"] == total_I and rep["particles"] == N
    assert seen.all()


def test_plan_x_slabs_balances_work():
    rng = np.random.default_rng(0)
    work = (rng.random(64) ** 4 * 1000 + 1).astype(np.int64).tolist()
    for world in (1, 2, 3, 4, 8):
        ranges = shard.plan_x_slabs(work, world)
        assert ranges[0][0] == 0 and ranges[-1][1] == 64
        assert all(a[1] == b[0] for a, b in zip(ranges, ranges[1:])) and all(hi > lo for lo, hi in ranges)
        loads = [sum(work[lo:hi]) for lo, hi in ranges]
        assert max(loads) <= sum(work) / world + max(work)
    assert shard.plan_x_slabs([0] * 5, 5) == [(i, i + 1) for i in range(5)]
    assert shard.plan_x_slabs([5, 0, 0, 0], 4) == [(0, 1), (1, 2), (2, 3), (3, 4)]
    with pytest.raises(ValueError):
        shard.plan_x_slabs([1, 2], 3)
    assert shard.ghost_sources(0, 4, 2, 8) == ([6, 7], [4, 5])
