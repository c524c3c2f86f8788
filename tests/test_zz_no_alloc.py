"""nf_timestep_terms_static -- the entry point that allocates nothing (scratch in a file-scope __device__ array,
include/nf.h) -- against the existing nf_timestep_terms on the same inputs, two calls in a row.  Collected last on purpose
(the suite runs with pytest -x).  Tolerances are those of test_gpu_parity.test_timestep_terms: minimum, maximum and counts
exact, the double sums within 1e-12."""
import ctypes

import numpy as np
import pytest
import torch

from paper_1810_02916_b200 import inputs

pytestmark = pytest.mark.gpu

EXACT = ("cells_used", "ratio_cell_min", "ratio_cell_max", "amax_global", "vmax")
ROUNDED = ("vrms_global", "ratio_global", "ratio_criterion2", "drift_limit")


@pytest.fixture(scope="module")
def ctx():
    from paper_1810_02916_b200 import nf
    c = nf.Context(0)
    yield c
    c.close()


def terms_inputs(ctx, n_side, K, seed):
    cfg = inputs.scaled(inputs.config(3), n_side ** 3, K)
    cfg = inputs.dataclasses.replace(cfg, n_halos=10, seed=seed)
    pos = inputs.make_positions(cfg, device="cuda")
    g = torch.Generator(device="cuda")
    g.manual_seed(seed)
    vel = torch.randn(cfg.N, 3, generator=g, device="cuda") * torch.exp(1.5 * torch.randn(cfg.N, 1, generator=g, device="cuda"))
    b = ctx.bin(pos, cfg.K, cfg.box)
    amax = torch.zeros(cfg.K ** 3, dtype=torch.float32, device="cuda")
    ctx.forces(b, cfg.R, cfg.eps, cfg.Gm, cell_amax=amax)
    vrms, vmax = ctx.cell_vrms(vel.contiguous(), b)
    return b, vrms, amax, vmax


def same(got, ref):
    for k in EXACT:
        assert got[k] == ref[k], (k, got[k], ref[k])
    for k in ROUNDED:
        assert abs(got[k] - ref[k]) <= 1e-12 * abs(ref[k]), (k, got[k], ref[k])


def test_static_scratch_matches_the_arena_path_two_calls_in_a_row(ctx):
    # first call: K = 20 -> 8000 cells, two records; second call: other inputs and K = 12 -> one record (the array still
    # holds the first call's second record: it must not be read)
    big = terms_inputs(ctx, 48, 20, 5)
    small = terms_inputs(ctx, 40, 12, 9)
    ref_big = ctx.timestep_terms(big[1], big[2], big[0], big[3])
    ref_small = ctx.timestep_terms(small[1], small[2], small[0], small[3])
    assert ref_big["cells_used"] > 4096 and ref_small["cells_used"] > 0
    got_big = ctx.timestep_terms_static(big[1], big[2], big[0], big[3])
    got_small = ctx.timestep_terms_static(small[1], small[2], small[0], small[3])
    same(got_big, ref_big)
    same(got_small, ref_small)
    # and again, the other way round; the same call gives the same bits every time
    assert ctx.timestep_terms_static(small[1], small[2], small[0], small[3]) == got_small
    assert ctx.timestep_terms_static(big[1], big[2], big[0], big[3]) == got_big
    assert ctx.timestep_terms_static(big[1], big[2], big[0])["drift_limit"] == float("inf")


def test_static_scratch_allocates_nothing_and_rejects_what_does_not_fit(ctx):
    from paper_1810_02916_b200 import nf
    b, vrms, amax, vmax = terms_inputs(ctx, 40, 12, 9)
    ctx.timestep_terms_static(vrms, amax, b, vmax)            # the symbol's address is looked up on the first call per device
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        ctx.timestep_terms_static(vrms, amax, b, vmax)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                       # no device memory was taken or returned
    # K beyond the array's capacity: refused before anything is read (the pointers are never dereferenced)
    ts = nf.TimeStep()
    rc = ctx.lib.nf_timestep_terms_static(ctx._h, vrms.data_ptr(), amax.data_ptr(), b.cell_offset.data_ptr(), 257, 1.0, None,
                                          ctypes.byref(ts), None)
    assert rc == nf.NF_ERR_ARG
    msg = ctx.lib.nf_last_error(ctx._h).decode()
    assert "static scratch" in msg and "256" in msg
    # the largest K it takes: 256^3 cells, 4096 records
    K = 256
    z = torch.zeros(K ** 3, dtype=torch.float32, device="cuda")
    off = torch.zeros(K ** 3 + 1, dtype=torch.int64, device="cuda")
    rc = ctx.lib.nf_timestep_terms_static(ctx._h, z.data_ptr(), z.data_ptr(), off.data_ptr(), K, 1.0, None, ctypes.byref(ts), None)
    assert rc == nf.NF_OK and ts.cells_used == 0 and ts.vrms_global == 0.0
