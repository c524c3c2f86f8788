#!/usr/bin/env python
"""bench.py -- the near-field force hot path (nf_bin + nf_forces) on seeded synthetic input.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

A "step" is one pass of the whole hot path (cell assignment,
histogram, scan, stable scatter + re-centre, work list, interaction kernel, scale/un-permute)
over one batch of synthetic particles.  The default workload is BASELINE.json's configs[3]
("C4", the clustered 1024^3 box the 60 % roofline target is quoted on); it fits one B200.

One JSON line is printed by rank 0 (DESIGN.md "Measurement" explains every key):
  value      pairwise interactions/s over the whole step, inputs resident in HBM
  e2e        the same through nf_forces_host: pinned HOST buffers, H2D + D2H inside the timing
  roofline   interaction kernel alone against the FP32 ALU peak, 20 flop per interaction
  cpu_baseline   the CPU oracle, as it stands, on a bounded sample of the same workload

`--config 5` is the slab-streaming workload (C5): a step is one nf_stream_slabs call over the
16 + 4 planes, from and to pinned host memory, so `value` already contains the copies.

`--impl reference` times the CPU oracle (this tier's reference arm) on bounded samples.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1810_02916_b200 import inputs  # noqa: E402

FLOP_PER_INTERACTION = 20          # BASELINE.json convention (the paper counts 23)
FP32_LANES_PER_SM = 128
ORACLE_BLOCK = 44                  # the oracle's sample is drawn from the sinks of a 44^3-cell block (~5 M sinks at 64 per cell)
ORACLE_SINKS = 1 << 22             # ... a seeded choice of this many of them, the SAME in both arms (cpu_baseline and --impl reference)
ORACLE_SEED = 1
ORACLE_MAX_PAIRS = 4e10            # ... cut back (the same way in both arms) when those sinks would mean more pairs than this (dense cells)


def ncu_traffic(workload: str):
    """roofline.traffic: dram bytes (read + write) of one interaction-kernel launch on `workload` from the ncu
    capture recorded in profiles/interaction_kernel_traffic.json by `python -m paper_1810_02916_b200.profiling
    traffic`, or None when that capture was taken from other kernel sources than the ones in this tree."""
    from paper_1810_02916_b200 import profiling
    return profiling.read_traffic(workload)


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return float(d.get("sm_max_mhz", 1965.0)), float(d.get("hbm_gbs", 6650.0)), "measured"
    return 1965.0, 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
            out, _ = self.p.communicate()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # "under load": samples in the upper half of the power range
        thr = 0.5 * (min(pw) + max(pw))
        load = [s for s, p in zip(sm, pw) if p >= thr] or sm
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(pos_dev: torch.Tensor, cfg, m: int, c0=(3, 5, 7)):
    """A block of m^3 sink cells with every source they need, for the CPU oracle: the particles
    whose coordinates lie within the block padded by R+1 cells (selected by coordinate range --
    the oracle does its own cell assignment with the full K and box)."""
    if cfg.K <= m + 2 * (cfg.R + 1):      # small box: hand the oracle everything
        return pos_dev.cpu().numpy(), None
    w = cfg.box / cfg.K
    lo = [(c - cfg.R - 1) * w for c in c0]
    hi = [(c + m + cfg.R + 1) * w for c in c0]
    idx = inputs.select_box(pos_dev, lo, hi, cfg.box)
    sub = pos_dev[idx].cpu().numpy()
    return sub, idx


def time_oracle(sub, cfg, m, c0, n_sinks=ORACLE_SINKS):
    """The oracle, as it stands, on a seeded sample of `n_sinks` sinks of the inner m^3 block (all their
    sources are in `sub`).  The SAME sample in both arms of the bench.  One oracle.forces call does its own
    cell assignment and sort of `sub` first (a fixed cost that does not scale with the sample); that part is
    timed by itself with oracle.bin_particles and reported beside the rate, which is pairs / (call - binning).
    Returns a dict: interactions, seconds (force part), seconds_binning, seconds_call, cores, n_sinks, sinks
    (indices into sub), acc (float64 [n_sinks, 3])."""
    import numpy as np
    import oracle
    K, R = cfg.K, cfg.R
    keys, _ = oracle.keys(sub, K, cfg.box)
    cz, cy, cx = keys % K, (keys // K) % K, keys // (K * K)
    inner = np.ones(len(keys), bool)
    for c, lo in ((cx, c0[0]), (cy, c0[1]), (cz, c0[2])):
        if K > m + 2 * (R + 1):
            inner &= ((c.astype(np.int64) - lo) % K) < m
    sink_idx = np.nonzero(inner)[0]
    rng = np.random.default_rng(ORACLE_SEED)
    timed = rng.choice(sink_idx, min(len(sink_idx), n_sinks), replace=False)
    cnt3 = np.bincount(keys, minlength=K ** 3).reshape(K, K, K).astype(np.int64)

    def pairs_of(sel):       # ordered pairs evaluated for the sinks `sel`, from the oracle's own cell counts
        kk = keys[sel].astype(np.int64)
        tz, ty, tx = kk % K, (kk // K) % K, kk // (K * K)
        tot = 0
        for dx in range(-R, R + 1):
            for dy in range(-R, R + 1):
                for dz in range(-R, R + 1):
                    tot += int(cnt3[(tx + dx) % K, (ty + dy) % K, (tz + dz) % K].sum())
        return tot

    inter = pairs_of(timed)
    if inter > ORACLE_MAX_PAIRS:
        timed = timed[: max(1, int(len(timed) * ORACLE_MAX_PAIRS / inter))]
        inter = pairs_of(timed)
    timed = np.sort(timed)
    t0 = time.perf_counter()
    oracle.bin_particles(sub, K, cfg.box)
    t_bin = time.perf_counter() - t0
    t0 = time.perf_counter()
    acc = oracle.forces(sub, K, R, cfg.eps, cfg.box, cfg.Gm, sink_idx=timed)
    t_call = time.perf_counter() - t0
    return {"interactions": inter, "seconds": max(t_call - t_bin, 1e-9), "seconds_binning": t_bin, "seconds_call": t_call,
            "cores": oracle.max_threads(), "n_sinks": len(timed), "sinks": timed, "acc": acc}


def cpu_baseline_block(o, cfg, m):
    return {"value": o["interactions"] / o["seconds"], "unit": "interactions/s", "cores": o["cores"], "kind": "oracle",
            "seconds": o["seconds"], "seconds_binning": o["seconds_binning"],
            "sample": f"{o['n_sinks']} seeded sinks of a {m}^3-cell block of {cfg.name} with all their sources "
                      f"({o['interactions']} pairs, float64); the oracle's own binning of the block ({o['seconds_binning']:.2f} s) "
                      f"is timed separately and not in the rate"}


def parity_block(a_gpu, a_ref):
    """GPU accelerations of the timed run against the oracle's, on the cpu_baseline sample: the north_star
    metric e = |da| / max(|a_ref|, rms |a_ref|) and the paper's own statistic, the fractional error
    |da| / |a| (median 7.5e-7, 0.038 % of particles above 1e-4 on the S2016 z = 0 state)."""
    import numpy as np
    import oracle
    a_gpu = np.asarray(a_gpu, dtype=np.float64)
    e = oracle.parity_error(a_gpu, a_ref)
    mag = np.sqrt((a_ref ** 2).sum(axis=1))
    fe = np.sqrt(((a_gpu - a_ref) ** 2).sum(axis=1)) / np.where(mag > 0, mag, 1.0)
    return {"n_sinks": int(e.size), "median": float(np.median(e)), "p999": float(np.quantile(e, 0.999)), "max": float(e.max()),
            "frac_err_median": float(np.median(fe)), "frac_gt_1e-4": float(np.mean(fe > 1e-4)),
            "tolerance": {"median": 1e-5, "max": 1e-3},
            "pass": bool(np.median(e) <= 1e-5 and e.max() <= 1e-3),
            "metric": "|a_gpu - a_ref| / max(|a_ref|, rms|a_ref|) over the sampled sinks; frac_err = |da|/|a| (PAPER.md:264)"}


def run_reference(args, cfg):
    """This tier's reference arm: the CPU oracle, as it stands, on the host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    m = ORACLE_BLOCK
    if cfg.kind == "slab":          # C5: the oracle is timed on the C4 box of the same recipe (same eps, halo catalogue, 64 per cell)
        cfg = inputs.config(4)
    pos = inputs.make_positions(cfg, device=dev)
    sub, _ = oracle_sample(pos, cfg, m)
    del pos
    per_step, o = [], None
    for it in range(args.warmup + args.steps):
        o = time_oracle(sub, cfg, m, (3, 5, 7))
        if it >= args.warmup:
            per_step.append(o["seconds"])
    ms = 1e3 * sum(per_step) / len(per_step)
    value = o["interactions"] / (ms * 1e-3)
    cb = cpu_baseline_block(o, cfg, m)
    cb["value"] = value
    line = {"impl": "reference", "metric": "near_field_pairwise_interactions_per_s", "value": value,
            "unit": "interactions/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "N": cfg.N, "K": cfg.K, "R": cfg.R, "eps": cfg.eps, "box": cfg.box},
            "cpu_baseline": cb,
            "e2e": {"value": value, "unit": "interactions/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_stream(args, cfg):
    """C5: nf_stream_slabs over P + 2R planes held in pinned host memory.
    One rank per GPU, every rank its own seeded chunk (weak scaling, no data-path collective)."""
    from paper_1810_02916_b200 import nf
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    rcfg = cfg if rank == 0 else inputs.dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)
    ctx = nf.Context(local)
    # particles are filed under the x-plane the library's own cell assignment gives them (nf_keys / K^2)
    plane_of = lambda x: ctx.keys(x.contiguous(), rcfg.K, rcfg.box).long() // (rcfg.K * rcfg.K)
    planes_dev = inputs.make_slab_planes(rcfg, device=dev, plane_of=plane_of)
    planes = []
    for t in planes_dev:
        h = torch.empty(t.shape, dtype=torch.float32).pin_memory()
        h.copy_(t)
        planes.append(h)
    del planes_dev, t
    torch.cuda.empty_cache()
    P, R, K = rcfg.planes, rcfg.R, rcfg.K
    n_in = sum(t.shape[0] for t in planes)
    n_out = sum(planes[R + p].shape[0] for p in range(P))
    Gm = 1.0 / float(rcfg.density_n) ** 3
    out = [torch.empty(planes[R + p].shape[0], 3, dtype=torch.float32).pin_memory() for p in range(P)]
    stats = None
    for _ in range(max(args.warmup, 1)):
        _, stats = ctx.stream_slabs(planes, P, K, R, rcfg.eps, rcfg.box, rcfg.plane0, Gm, out=out)
    I = stats["interactions"]
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    all_stats = []
    barrier()
    t0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        _, st = ctx.stream_slabs(planes, P, K, R, rcfg.eps, rcfg.box, rcfg.plane0, Gm, out=out)
        all_stats.append(st)
    e1.record()
    barrier()
    wall = time.perf_counter() - t0
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop() if sampler else None
    t = torch.tensor([max(wall, e0.elapsed_time(e1) * 1e-3)], dtype=torch.float64, device=dev)
    tot = torch.tensor([float(I), float(n_out)], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    ms_per_step = 1e3 * float(t.item()) / args.steps
    value = float(tot[0].item()) / (ms_per_step * 1e-3)
    mean = lambda k: sum(s[k] for s in all_stats) / len(all_stats)
    sm_max_mhz, hbm_gbs, peak_src = read_peaks()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak_tflops = sms * sm_max_mhz * 1e6 * 2 * FP32_LANES_PER_SM / 1e12
    f_ms = 1e3 * mean("force_seconds")
    achieved = FLOP_PER_INTERACTION * I / (f_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": "interaction kernel (16 launches, one per sink plane, with their work-list kernels)",
                "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                "traffic": ncu_traffic(rcfg.name),
                "peak_source": f"{sms} SMs x {sm_max_mhz:.0f} MHz ({peak_src} sm_max_mhz) x 2 x {FP32_LANES_PER_SM} FP32 lanes",
                "flop_per_interaction": FLOP_PER_INTERACTION, "frac_at_paper_23_flop": achieved / peak_tflops * 23.0 / FLOP_PER_INTERACTION,
                "kernel_ms": f_ms,
                "kernel_interactions_per_s": I / (f_ms * 1e-3), "kernel_share_of_step": f_ms / ms_per_step}
    e2e = {"value": value, "unit": "interactions/s", "h2d_bytes_per_step": int(mean("h2d_bytes")),
           "d2h_bytes_per_step": int(mean("d2h_bytes")), "ms_per_step": ms_per_step, "api": "nf_stream_slabs",
           "note": "this workload lives in pinned host memory by definition: value and e2e are the same measurement",
           "result_checksum": float(sum(float(o[:: max(1, o.shape[0] // 256)].double().abs().sum()) for o in out))}
    copies = {"h2d_gbps": mean("h2d_gbps"), "d2h_gbps": mean("d2h_gbps"), "overlap_fraction": mean("overlap_fraction"),
              "h2d_seconds": mean("h2d_seconds"), "d2h_seconds": mean("d2h_seconds"),
              "kernel_seconds": mean("kernel_seconds"), "wall_seconds": mean("wall_seconds")}
    line = {"metric": "near_field_pairwise_interactions_per_s", "value": value, "unit": "interactions/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": rcfg.name, "planes": P, "ghost_planes": 2 * R, "K": K, "R": R, "eps": rcfg.eps,
                       "box": rcfg.box, "particles_in": n_in, "particles_out": n_out,
                       "interactions_per_step_per_gpu": I, "interactions_per_particle": I / max(n_out, 1),
                       "l2": "inputs larger than L2 (streamed from pinned host memory)",
                       "parallelism": f"{world} independent chunks, one per GPU" if world > 1 else "1 GPU"},
            "particles_per_s": float(tot[1].item()) / (ms_per_step * 1e-3),
            "e2e": e2e, "copies": copies, "gpu_launches": launches, "clocks": clocks, "roofline": roofline,
            "cpu_baseline": None}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def run_sharded(args, cfg):
    """N > 1 GPUs: ONE box of the named config cut into N contiguous x-slab ranges balanced by pairwise
    interactions (SURVEY.md Sec. 8(e); PAPER.md:41 slabs, :81 "a parallel version of Abacus based on the
    existing slab decomposition").  A rank holds the particles of its planes, filed by plane.  One step =
    ONE exchange of R ghost planes with each x-neighbour (point-to-point, no all-reduce, no output
    exchange) + nf_bin + nf_forces_chunk on (own + ghost) particles; all of it inside the timed region.
    Strong scaling: the total work is fixed as N grows.  Also runs with N = 1 (`--shard`), where the
    single range is the whole periodic box and there is nothing to exchange."""
    from paper_1810_02916_b200 import nf, shard
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    same_gpu = args.shard_backend == "gloo"          # debugging aid: every rank on cuda:0, ghosts staged through the host
    local = 0 if same_gpu else local
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        if same_gpu:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    K, R, N = cfg.K, cfg.R, cfg.N
    KK = K * K
    ctx = nf.Context(local)
    n_chunks = (N + inputs.CHUNK - 1) // inputs.CHUNK
    # ---- the plan: per-plane work from the box's cell counts (each rank counts 1/world of the chunks)
    cnt = torch.zeros(K ** 3, dtype=torch.int64, device=dev)
    for c in range(rank, n_chunks, world):
        x = inputs.make_positions_chunk(cfg, c, device=dev)
        cnt += torch.bincount(ctx.keys(x, K, cfg.box).long(), minlength=K ** 3)
    if world > 1:
        if same_gpu:
            h = cnt.cpu()
            dist.all_reduce(h)
            cnt.copy_(h)
        else:
            dist.all_reduce(cnt)
    c3 = cnt.view(K, K, K)
    nb = torch.zeros_like(c3)
    for dx in range(-R, R + 1):
        for dy in range(-R, R + 1):
            for dz in range(-R, R + 1):
                nb += torch.roll(c3, shifts=(dx, dy, dz), dims=(0, 1, 2))
    work = (c3 * nb).sum(dim=(1, 2)).tolist()          # ordered pairs whose sink lies in plane p
    I_total = int(sum(work))
    ranges = shard.plan_x_slabs(work, world)
    lo, hi = ranges[rank]
    ghosts = shard.ghost_planes(lo, hi, R, K) if world > 1 else []
    if world > 1 and any(h - l + 2 * R > K for l, h in ranges):
        raise SystemExit("bench.py: a rank's planes plus ghosts exceed the box (K too small for this many ranks)")
    plane_n = c3.sum(dim=(1, 2)).tolist()
    n_own = int(sum(plane_n[lo:hi]))
    n_ghost = int(sum(plane_n[p] for p in ghosts))
    del cnt, c3, nb
    # ---- this rank's particles, filed by plane (stable), with room for the ghosts behind them
    local_pos = torch.empty(n_own + n_ghost, 3, dtype=torch.float32, device=dev)
    plane_id = torch.empty(n_own, dtype=torch.int64, device=dev)
    fill = 0
    for c in range(n_chunks):
        x = inputs.make_positions_chunk(cfg, c, device=dev)
        p = ctx.keys(x, K, cfg.box).long() // KK
        keep = (p >= lo) & (p < hi)
        m = int(keep.sum())
        local_pos[fill:fill + m] = x[keep]
        plane_id[fill:fill + m] = p[keep]
        fill += m
    assert fill == n_own
    order = torch.argsort(plane_id, stable=True)
    local_pos[:n_own] = local_pos[:n_own][order]
    del order, plane_id, x, p, keep
    starts = [0]
    for q in range(lo, hi):
        starts.append(starts[-1] + int(plane_n[q]))
    my_planes = [local_pos[starts[i]:starts[i + 1]] for i in range(hi - lo)]
    need_l, need_r = shard.ghost_sources(lo, hi, R, K)
    slot_plane = need_l + need_r
    goff, o = {}, n_own
    for pl in ghosts:
        goff[pl] = o
        o += int(plane_n[pl])

    def alloc(slot, n):
        pl = slot_plane[slot]
        assert n == int(plane_n[pl])
        return local_pos[goff[pl]:goff[pl] + n]

    torch.cuda.empty_cache()
    ctx.reserve(n_own + n_ghost, K)
    b = None
    acc = torch.empty(n_own + n_ghost, 3, dtype=torch.float32, device=dev)

    def step():
        nonlocal b
        if world > 1:
            shard.exchange_ghosts(my_planes, ranges, R, K, dist, rank=rank, alloc=alloc, via_host=same_gpu)
        b = ctx.bin(local_pos, K, cfg.box, out=b)
        ctx.forces_chunk(b, R, cfg.eps, cfg.Gm, lo, hi, out=acc)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = ctx.launch_count()
    kern_ms = []
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e0.record()
    for s_ in range(args.steps):
        step()
        kern_ms.append(ctx.last_forces_timing()[0])
    e1.record()
    barrier()
    wall = time.perf_counter() - t0
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop() if sampler else None
    k_ms = sum(kern_ms) / len(kern_ms)
    red = lambda v, op: v
    t = torch.tensor([max(wall, e0.elapsed_time(e1) * 1e-3), k_ms * 1e-3], dtype=torch.float64)
    if world > 1:
        t = t if same_gpu else t.to(dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_per_step = 1e3 * float(t[0]) / args.steps
    k_ms_max = 1e3 * float(t[1])

    # ---- end to end: own particles from pinned host memory, accelerations back to it, every step
    e2e = None
    if not args.no_e2e:
        h_own = torch.empty(n_own, 3, dtype=torch.float32).pin_memory()
        h_own.copy_(local_pos[:n_own])
        h_acc = torch.empty(n_own, 3, dtype=torch.float32).pin_memory()
        n_e2e = max(1, min(args.steps, 3))

        def e2e_step():
            local_pos[:n_own].copy_(h_own, non_blocking=True)
            step()
            h_acc.copy_(acc[:n_own], non_blocking=True)
            torch.cuda.synchronize()

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        barrier()
        te = torch.tensor([(time.perf_counter() - t0) / n_e2e], dtype=torch.float64)
        if world > 1:
            te = te if same_gpu else te.to(dev)
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": I_total / float(te[0]), "unit": "interactions/s", "h2d_bytes_per_step": 12 * N, "d2h_bytes_per_step": 12 * N,
               "ms_per_step": 1e3 * float(te[0]), "api": "H2D own planes + ghost exchange + nf_bin + nf_forces_chunk + D2H", "steps": n_e2e,
               "result_checksum": float(h_acc[:: max(1, n_own // 4096)].double().abs().sum())}

    # parity of rank 0's sinks against the oracle on a block inside its range (N = 1: --shard only)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    value = I_total / (ms_per_step * 1e-3)
    sm_max_mhz, hbm_gbs, peak_src = read_peaks()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak_tflops = world * sms * sm_max_mhz * 1e6 * 2 * FP32_LANES_PER_SM / 1e12
    achieved = FLOP_PER_INTERACTION * I_total / (k_ms_max * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": "interaction kernel (nf_forces_chunk), slowest rank", "achieved": achieved, "peak": peak_tflops,
                "unit": "TFLOP/s", "frac": achieved / peak_tflops, "traffic": None,
                "peak_source": f"{world} x {sms} SMs x {sm_max_mhz:.0f} MHz ({peak_src} sm_max_mhz) x 2 x {FP32_LANES_PER_SM} FP32 lanes",
                "flop_per_interaction": FLOP_PER_INTERACTION, "kernel_ms": k_ms_max, "kernel_share_of_step": k_ms_max / ms_per_step}
    line = {"metric": "near_field_pairwise_interactions_per_s", "value": value, "unit": "interactions/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
            "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "N": N, "K": K, "R": R, "eps": cfg.eps, "box": cfg.box,
                       "interactions_per_step": I_total, "interactions_per_particle": I_total / N,
                       "l2": "inputs larger than L2",
                       "parallelism": f"x-slab sharding over {world} GPU(s), R ghost planes from each x-neighbour, ranges balanced by interactions",
                       "ranges": ranges, "rank0_particles": n_own, "rank0_ghost_particles": n_ghost,
                       "ghost_bytes_per_step_rank0": 12 * n_ghost},
            "particles_per_s": N / (ms_per_step * 1e-3),
            "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": None}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_tree(args, cfg):
    """`--tree THETA`: the step with nf_forces_tree in place of nf_forces.
    One GPU.  `value` counts the interactions the step EVALUATED (pairs of the interaction kernel for the sources that are
    not in dense cells + (sink, particle of an opened leaf) + (sink, accepted node)); the direct sum's pair count of the
    same box and the time of the direct step are reported beside it."""
    import numpy as np
    from paper_1810_02916_b200 import nf
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(0)
    theta = float(args.tree)
    ctx = nf.Context(0)
    pos = inputs.make_positions(cfg, device=dev)
    N, K, R = cfg.N, cfg.K, cfg.R
    b = ctx.bin(pos, K, cfg.box)
    acc = torch.empty(N, 3, dtype=torch.float32, device=dev)
    I_direct = ctx.interactions(b, R)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if N * 28 < (256 << 20) else None

    def step_tree():
        ctx.bin(pos, K, cfg.box, out=b)
        ctx.forces_tree(b, R, cfg.eps, cfg.Gm, theta, out=acc)

    def step_direct():
        ctx.bin(pos, K, cfg.box, out=b)
        ctx.forces(b, R, cfg.eps, cfg.Gm, out=acc)

    def timed(step, steps, want_walk):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        walk, kern = [], []
        torch.cuda.synchronize()
        for s_ in range(steps):
            if flush is not None:
                flush.fill_(s_)
            ev[s_][0].record()
            step()
            ev[s_][1].record()
            kern.append(ctx.last_forces_timing()[0])
            if want_walk:
                walk.append(ctx.last_tree_timing())
        torch.cuda.synchronize()
        return sum(a.elapsed_time(c) for a, c in ev) / steps, sum(kern) / steps, (sum(walk) / steps if walk else None)

    for _ in range(args.warmup):
        step_direct()
    direct_ms, direct_k_ms, _ = timed(step_direct, args.steps, False)
    a_direct = acc.clone()
    for _ in range(args.warmup):
        step_tree()
    sampler = ClockSampler(0)
    launches0 = ctx.launch_count()
    ms_per_step, k_ms, walk_ms = timed(step_tree, args.steps, True)
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop()
    st = ctx.tree_stats()
    # pairs the interaction kernel still evaluated: sources of cells below the dense threshold (reading t1)
    cnt = b.cell_count.cpu().numpy().astype(np.int64).reshape(K, K, K)
    coff, rank, dense = 0, 0, np.zeros(K ** 3, dtype=bool)
    cap = min(max(N, 1 << 20) + 64 * 2048, 1 << 28) & ~63
    for c, n in enumerate(cnt.ravel()):
        if n >= 4096:
            n64 = (int(n) + 63) & ~63
            dense[c] = rank < 2048 and coff + n64 <= cap
            coff += n64
            rank += 1
    light = np.where(dense.reshape(K, K, K), 0, cnt)
    I_kernel = 0
    for d in np.ndindex(2 * R + 1, 2 * R + 1, 2 * R + 1):
        I_kernel += int((cnt * np.roll(light, shift=(R - d[0], R - d[1], R - d[2]), axis=(0, 1, 2))).sum())
    I_eval = I_kernel + st["node"] + st["leaf"]
    value = I_eval / (ms_per_step * 1e-3)
    # how far the approximation is from the direct sum (both on the GPU, all sinks)
    mag = a_direct.double().norm(dim=1)
    err = (acc.double() - a_direct.double()).norm(dim=1) / torch.maximum(mag, mag.pow(2).mean().sqrt())
    approx = {"against": "nf_forces of the same box (direct sum), all sinks", "median": float(err.median()),
              "p99": float(err.kthvalue(int(0.99 * N)).values), "max": float(err.max())}
    # ---- end to end: positions from pinned host memory, accelerations back into pinned host memory ----
    e2e = None
    if not args.no_e2e:
        hpos = torch.empty(N, 3, dtype=torch.float32, pin_memory=True).copy_(pos)
        hacc = torch.empty(N, 3, dtype=torch.float32, pin_memory=True)
        dpos = torch.empty_like(pos)

        def host_step():
            dpos.copy_(hpos, non_blocking=True)
            ctx.bin(dpos, K, cfg.box, out=b)
            ctx.forces_tree(b, R, cfg.eps, cfg.Gm, theta, out=acc)
            hacc.copy_(acc, non_blocking=True)
            torch.cuda.synchronize()

        host_step()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            host_step()
        e_s = (time.perf_counter() - t0) / args.steps
        e2e = {"value": I_eval / e_s, "unit": "interactions/s", "h2d_bytes_per_step": 12 * N, "d2h_bytes_per_step": 12 * N,
               "ms_per_step": 1e3 * e_s, "api": "Context.bin + Context.forces_tree on positions copied from pinned host memory, accelerations copied back",
               "result_checksum": float(hacc[:: max(1, N // 4096)].double().abs().sum())}
    sm_max_mhz, hbm_gbs, peak_src = read_peaks()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak_tflops = sms * sm_max_mhz * 1e6 * 2 * FP32_LANES_PER_SM / 1e12
    achieved = FLOP_PER_INTERACTION * (st["node"] + st["leaf"]) / (walk_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": "tree walk (k_tree_walk)", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved / peak_tflops, "traffic": None,
                "peak_source": f"{sms} SMs x {sm_max_mhz:.0f} MHz ({peak_src} sm_max_mhz) x 2 x {FP32_LANES_PER_SM} FP32 lanes",
                "flop_per_interaction": FLOP_PER_INTERACTION, "kernel_ms": walk_ms, "kernel_share_of_step": walk_ms / ms_per_step,
                "interaction_kernel_ms": k_ms,
                "note": "node and leaf interactions both counted at the direct kernel's flop per interaction; the walk also tests boxes and moves a stack"}
    cpu, parity = None, None
    if not args.no_cpu:
        from oracle import nf_tree
        pos_np = pos.cpu().numpy()
        sinks = np.sort(np.random.default_rng(ORACLE_SEED).choice(N, min(N, 384), replace=False))
        t0 = time.perf_counter()
        ref = nf_tree.forces_tree(pos_np, K, R, cfg.eps, cfg.box, cfg.Gm, theta, sink_idx=sinks)
        sec = time.perf_counter() - t0
        parity = parity_block(acc[torch.from_numpy(sinks).to(dev)].cpu().numpy(), ref)
        cpu = {"value": len(sinks) * (I_eval / N) / sec, "unit": "interactions/s", "cores": 1, "kind": "oracle", "seconds": sec,
               "sample": f"oracle/nf_tree.py forces_tree (numpy, one process) for {len(sinks)} seeded sinks of {cfg.name} -- every 64-sink group "
                         f"that holds one of them is walked and summed; rate = sinks x mean evaluated interactions per sink / seconds"}
    line = {"metric": "near_field_pairwise_interactions_per_s", "value": value, "unit": "interactions/s", "n_gpus": 1,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name + f" + tree theta={theta:g}", "N": N, "K": K, "R": R, "eps": cfg.eps, "box": cfg.box,
                       "theta": theta, "interactions_per_step_per_gpu": I_eval,
                       "l2": "flushed between timed steps (256 MiB write)" if flush is not None else "inputs larger than L2",
                       "parallelism": "1 GPU"},
            "tree": {"theta": theta, "node_interactions": st["node"], "leaf_interactions": st["leaf"], "interaction_kernel_pairs": I_kernel,
                     "direct_sum_pairs": I_direct, "direct_step_ms": direct_ms, "speedup_over_direct_step": direct_ms / ms_per_step,
                     "direct_equivalent_interactions_per_s": I_direct / (ms_per_step * 1e-3), "walk_ms": walk_ms,
                     "approximation_error": approx},
            "particles_per_s": N / (ms_per_step * 1e-3), "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
            "roofline": roofline, "cpu_baseline": cpu, "parity": parity, "sweep": None}
    print(json.dumps(line), flush=True)


def run_occupancy(args):
    """`--occupancy`: the interaction kernel on boxes whose cells ALL hold exactly n particles (uniform inside the cell), K = 48,
    R = 2: kernel time and fraction of the FP32 roofline as a function of the occupancy, i.e. of the task shape (L = ceil(n/4)
    lanes, P = floor(32/L) phases) and of the tile length (5n sources per column).  A measuring aid for DESIGN.md Sec. 11."""
    from paper_1810_02916_b200 import nf
    dev = torch.device("cuda", 0)
    ctx = nf.Context(0)
    K, R, box = 48, 2, 1.0
    w = box / K
    g = torch.Generator(device=dev)
    g.manual_seed(5)
    cells = torch.stack(torch.meshgrid(torch.arange(K), torch.arange(K), torch.arange(K), indexing="ij"), -1).reshape(-1, 3).to(dev).float()
    sm_max_mhz, _, peak_src = read_peaks()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak = sms * sm_max_mhz * 1e6 * 2 * FP32_LANES_PER_SM
    rows = []
    for n in (4, 8, 12, 16, 20, 24, 28, 32, 36, 40, 44, 48, 52, 56, 60, 64, 72, 80, 96, 112, 128):
        pos = ((cells[:, None, :] + 0.02 + 0.96 * torch.rand(K ** 3, n, 3, generator=g, device=dev)) * w).reshape(-1, 3).contiguous()
        b = ctx.bin(pos, K, box)
        I = ctx.interactions(b, R)
        ts = []
        for s_ in range(args.warmup + args.steps):
            ctx.forces(b, R, 0.01 * w, 1.0)
            if s_ >= args.warmup:
                ts.append(ctx.last_forces_timing()[0])
        k_ms = statistics.median(ts)
        rows.append({"n": n, "kernel_ms": k_ms, "frac": FLOP_PER_INTERACTION * I / (k_ms * 1e-3) / peak})
    print(json.dumps({"occupancy_sweep": rows, "K": K, "R": R, "peak_source": f"{sms} SMs x {sm_max_mhz:.0f} MHz ({peak_src})"}), flush=True)


def sweep_small_configs(ctx, dev, steps=3, warmup=3):
    """Interaction-kernel roofline fraction of C1, C2 and C3 -- the other single-GPU configs of BASELINE.json beside the
    headline workload -- and of D1, the one-dense-cell workload (config 6), in the same process (milliseconds each).  Same timing rules as the main
    line: W warm-up steps, the L2 flushed between timed steps (inputs smaller than the L2), CUDA events
    around the kernel inside nf_forces."""
    sm_max_mhz, _, _ = read_peaks()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak = sms * sm_max_mhz * 1e6 * 2 * FP32_LANES_PER_SM
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    out = {}
    for which in (1, 2, 3, 6):
        cfg = inputs.config(which)
        pos = inputs.make_positions(cfg, device=dev)
        b = ctx.bin(pos, cfg.K, cfg.box)
        acc = torch.empty(cfg.N, 3, dtype=torch.float32, device=dev)
        I = ctx.interactions(b, cfg.R)
        k_ms, s_ms = [], []
        for it in range(warmup + steps):
            flush.fill_(it)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.bin(pos, cfg.K, cfg.box, out=b)
            ctx.forces(b, cfg.R, cfg.eps, cfg.Gm, out=acc)
            e1.record()
            k = ctx.last_forces_timing()[0]
            if it >= warmup:
                k_ms.append(k)
                s_ms.append(e0.elapsed_time(e1))
        k = sum(k_ms) / len(k_ms)
        graph_ms = None
        if which == 1:
            # the smallest config is launch-bound (~45 launches for 0.3 ms of kernels): the same step replayed from a CUDA graph
            try:
                st = torch.cuda.Stream()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.stream(st):
                    ctx.bin(pos, cfg.K, cfg.box, out=b, stream=st)
                    ctx.forces(b, cfg.R, cfg.eps, cfg.Gm, out=acc, stream=st)
                    st.synchronize()
                    g.capture_begin()
                    ctx.bin(pos, cfg.K, cfg.box, out=b, stream=st)
                    ctx.forces(b, cfg.R, cfg.eps, cfg.Gm, out=acc, stream=st)
                    g.capture_end()
                torch.cuda.synchronize()
                g.replay()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                for _ in range(20):
                    g.replay()
                e1.record()
                torch.cuda.synchronize()
                graph_ms = e0.elapsed_time(e1) / 20
                del g
            except Exception:
                graph_ms = None
        out[cfg.name] = {"kernel_ms": k, "step_ms": sum(s_ms) / len(s_ms), "step_ms_cuda_graph": graph_ms, "interactions": I,
                         "frac": FLOP_PER_INTERACTION * I / (k * 1e-3) / peak,
                         "interactions_per_s_step": I / (sum(s_ms) / len(s_ms) * 1e-3)}
        del pos, b, acc
    del flush
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number 1..5 (default 4 = C4; 5 = slab streaming); 6 = one dense cell of 4x10^5 particles (profiling workload); 7 = the C3 recipe at K = 16: 254 dense cells (for --tree)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip the C1-C3 + D1 kernel sweep of the default line")
    ap.add_argument("--shard", action="store_true", help="use the x-slab sharded path (the default for --gpus N > 1) even on one GPU")
    ap.add_argument("--shard-backend", default="nccl", choices=["nccl", "gloo"],
                    help="gloo: debugging aid, every rank on cuda:0 with ghosts staged through host memory")
    ap.add_argument("--n-side", type=int, default=0,
                    help="profiling aid: the same recipe at n_side^3 particles and K = n_side/4 (not the bench workload)")
    ap.add_argument("--occupancy", action="store_true",
                    help="measuring aid: kernel efficiency on boxes whose cells all hold exactly n particles, n = 4 ... 128")
    ap.add_argument("--tree", type=float, default=None, metavar="THETA",
                    help="time the step with nf_forces_tree (tree near field for dense cells, opening angle THETA) instead of nf_forces")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = max(args.warmup, 0)
    cfg = inputs.config(args.config)
    if args.n_side:
        cfg = inputs.scaled(cfg, args.n_side ** 3, args.n_side // 4)

    if args.impl == "reference":
        run_reference(args, cfg)
        return

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    if cfg.kind == "slab":
        run_stream(args, cfg)
        return
    if args.occupancy:
        run_occupancy(args)
        return
    if args.tree is not None:
        if int(os.environ.get("WORLD_SIZE", "1")) > 1:
            raise SystemExit("bench.py --tree: one GPU (the tree near field takes a whole box)")
        run_tree(args, cfg)
        return
    if args.shard or int(os.environ.get("WORLD_SIZE", "1")) > 1:
        run_sharded(args, cfg)
        return
    from paper_1810_02916_b200 import nf

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # every rank owns an independently seeded box of the same recipe (weak scaling)
    rcfg = cfg if rank == 0 else inputs.dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)
    ctx = nf.Context(local)
    sweep = None
    if args.config == 4 and not args.n_side and not args.no_sweep and world == 1:
        sweep = sweep_small_configs(ctx, dev)
    pos = inputs.make_positions(rcfg, device=dev)
    N, K, R = rcfg.N, rcfg.K, rcfg.R
    ctx.reserve(N, K)
    b = ctx.bin(pos, K, rcfg.box)
    acc = torch.empty(N, 3, dtype=torch.float32, device=dev)
    I = ctx.interactions(b, R)
    flush = None
    small = N * 28 < (256 << 20)
    if small:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step():
        ctx.bin(pos, K, rcfg.box, out=b)
        ctx.forces(b, R, rcfg.eps, rcfg.Gm, out=acc)

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    launches0 = ctx.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms = []
    barrier()
    for s in range(args.steps):
        if flush is not None:
            flush.fill_(s)
        ev[s][0].record()
        step()
        ev[s][1].record()
        kern_ms.append(ctx.last_forces_timing()[0])   # synchronises on the step's end event
    barrier()
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop() if sampler else None
    step_ms = [a.elapsed_time(bb) for a, bb in ev]
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device=dev)
    I_all = torch.tensor([float(I)], dtype=torch.float64, device=dev)
    N_all = torch.tensor([float(N)], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
        dist.all_reduce(I_all)
        dist.all_reduce(N_all)
    ms_per_step = float(total_ms.item()) / args.steps
    value = float(I_all.item()) / (ms_per_step * 1e-3)
    k_ms = sum(kern_ms) / len(kern_ms)

    # sample for the CPU oracle (taken now, while the positions and the accelerations of the last timed
    # step are still on the device): the block's particles, and the GPU's accelerations of the same rows
    cpu_sub, acc_sub = None, None
    if not args.no_cpu and world == 1 and rank == 0:
        cpu_sub, sub_idx = oracle_sample(pos, rcfg, ORACLE_BLOCK)
        acc_sub = (acc if sub_idx is None else acc[sub_idx]).cpu().numpy()
        del sub_idx

    # ---- end to end through nf_forces_host (pinned host buffers, copies inside the timing) ----
    e2e = None
    if not args.no_e2e:
        try:
            import psutil
            need = 36 * N * world * 1.15            # pinned host input + two outputs of every rank on this node
            if psutil.virtual_memory().available < need:
                raise MemoryError(f"host leg needs {need / 2**30:.0f} GiB of pinned memory for {world} rank(s)")
            del b, acc
            torch.cuda.empty_cache()
            hpos = torch.empty(N, 3, dtype=torch.float32).pin_memory()
            hpos.copy_(pos)
            del pos
            torch.cuda.empty_cache()
            hacc = [torch.empty(N, 3, dtype=torch.float32).pin_memory() for _ in range(2)]
            # (a) one blocking call per step: H2D, compute, D2H in sequence -- the latency of ONE step end to end
            ctx.reserve_host(N, K)
            ctx.forces_host(hpos, K, R, rcfg.eps, rcfg.box, rcfg.Gm, out=hacc[0])
            barrier()
            t0 = time.perf_counter()
            ctx.forces_host(hpos, K, R, rcfg.eps, rcfg.box, rcfg.Gm, out=hacc[0])
            barrier()
            serial_s = time.perf_counter() - t0
            # (b) the two-deep pipeline nf_forces_host_begin / _end: step s+1's H2D and step s's D2H run behind the
            # kernels of the step in between.  Timed in steady state: every iteration completes one whole step
            # (whose H2D, kernels and D2H all ran inside the timed region or overlapped the previous iteration's).
            # (long steps: 3-5 of them; short steps: as many as fill half a second, so that the few-step noise of the host clock
            # does not decide the number -- C2 read 7.56 ms over 5 steps and 7.06 ms over 20)
            n_e2e = max(3, min(args.steps, 5)) if ms_per_step > 100.0 else min(50, max(5, int(500.0 / max(ms_per_step, 1e-3))))
            ctx.forces_host_begin(hpos, K, R, rcfg.eps, rcfg.box, rcfg.Gm, hacc[0])
            ctx.forces_host_begin(hpos, K, R, rcfg.eps, rcfg.box, rcfg.Gm, hacc[1])
            ctx.forces_host_end()                                   # the pipeline is primed: one step in flight
            t0 = time.perf_counter()
            for s_ in range(n_e2e):
                ctx.forces_host_begin(hpos, K, R, rcfg.eps, rcfg.box, rcfg.Gm, hacc[s_ % 2])
                ctx.forces_host_end()
            wall = (time.perf_counter() - t0) / n_e2e
            ctx.forces_host_end()                                   # drain
            barrier()
            t = torch.tensor([wall], dtype=torch.float64, device=dev)
            if dist is not None:
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e = {"value": float(I_all.item()) / float(t.item()), "unit": "interactions/s",
                   "h2d_bytes_per_step": 12 * N, "d2h_bytes_per_step": 12 * N,
                   "ms_per_step": 1e3 * float(t.item()), "api": "nf_forces_host_begin / nf_forces_host_end (two steps in flight)",
                   "steps": n_e2e, "timing": "host wall clock over completed steps in steady state (each end() returns after that step's D2H)",
                   "single_call_ms": 1e3 * serial_s, "single_call_api": "nf_forces_host (H2D, kernels, D2H in sequence)",
                   "single_call_value": float(I) / serial_s,
                   "copies_hidden_fraction": max(0.0, min(1.0, (serial_s - float(t.item())) / max(serial_s - ms_per_step * 1e-3, 1e-9))),
                   "result_checksum": float(hacc[0][:: max(1, N // 4096)].double().abs().sum())}
        except Exception as exc:  # keep the device-timed line even if the host leg cannot run
            e2e = {"value": None, "unit": "interactions/s", "error": repr(exc)[:200]}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    sm_max_mhz, hbm_gbs, peak_src = read_peaks()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak_tflops = sms * sm_max_mhz * 1e6 * 2 * FP32_LANES_PER_SM / 1e12
    achieved = FLOP_PER_INTERACTION * I / (k_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": "interaction kernel (nf_forces)", "achieved": achieved,
                "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops, "traffic": ncu_traffic(rcfg.name),
                "peak_source": f"{sms} SMs x {sm_max_mhz:.0f} MHz ({peak_src} sm_max_mhz) x 2 x {FP32_LANES_PER_SM} FP32 lanes",
                "flop_per_interaction": FLOP_PER_INTERACTION, "frac_at_paper_23_flop": achieved / peak_tflops * 23.0 / FLOP_PER_INTERACTION,
                "kernel_ms": k_ms,
                "kernel_interactions_per_s": I / (k_ms * 1e-3), "kernel_share_of_step": k_ms / ms_per_step,
                "frac_at_sampled_clock": (achieved / (peak_tflops * clocks["sm_mhz"] / sm_max_mhz)
                                          if clocks and clocks.get("sm_mhz") else None)}

    cpu, parity = None, None
    if cpu_sub is not None:
        o = time_oracle(cpu_sub, rcfg, ORACLE_BLOCK, (3, 5, 7))
        cpu = cpu_baseline_block(o, rcfg, ORACLE_BLOCK)
        # the oracle's accelerations of the timed sample against the GPU's from the last TIMED step
        parity = parity_block(acc_sub[o["sinks"]], o["acc"])

    line = {"metric": "near_field_pairwise_interactions_per_s", "value": value, "unit": "interactions/s",
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": rcfg.name, "N": N, "K": K, "R": R, "eps": rcfg.eps, "box": rcfg.box,
                       "interactions_per_step_per_gpu": I, "interactions_per_particle": I / N,
                       "l2": "flushed between timed steps (256 MiB write)" if small else "inputs larger than L2",
                       "parallelism": f"{world} independent boxes, one per GPU" if world > 1 else "1 GPU"},
            "particles_per_s": float(N_all.item()) / (ms_per_step * 1e-3),
            "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
            "parity": parity, "sweep": sweep}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
