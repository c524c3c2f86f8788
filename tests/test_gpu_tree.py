"""Parity of the tree near field for dense cells (nf_forces_tree; readings t1-t6) against its CPU
oracle (oracle/nf_tree.py) through the C ABI.  The walk's decisions are float32 in a fixed order of rounded operations on
both sides, so the interaction counts are compared bit for bit and the accelerations within the usual bars."""
import numpy as np
import pytest
import torch

import oracle
from oracle import nf_tree
from paper_1810_02916_b200 import inputs

pytestmark = pytest.mark.gpu

MEDIAN_TOL = 1e-5
MAX_TOL = 1e-3


@pytest.fixture(scope="module")
def ctx():
    from paper_1810_02916_b200 import nf
    c = nf.Context(0)
    yield c
    c.close()


CASES = {
    # K, R, box, eps, clumps, background
    "three-clumps-R1": (4, 1, 4.0, 0.02, [((1, 1, 1), 4500, 0.3, (0.1, 0, 0)), ((1, 1, 2), 4200, 0.45, (0, 0, -0.05)),
                                          ((3, 0, 1), 4100, 0.2, (0, 0.2, 0))], 1500),
    "two-clumps-R2-wrap": (5, 2, 1.0, 0.002, [((0, 0, 0), 9000, 0.5, (0, 0, 0)), ((4, 4, 3), 5000, 0.25, (0.2, 0.2, 0))], 3000),
    # every source of every sink is in a dense cell: the interaction kernel is left with sentinel tiles only
    "dense-only": (3, 1, 3.0, 0.01, [((1, 1, 1), 6000, 0.4, (0, 0, 0)), ((1, 2, 1), 4096, 0.3, (0, -0.1, 0))], 0),
    # a ragged big cell: 3 levels above the leaves, last leaf of 1 particle
    "one-big-cell": (3, 1, 3.0, 0.005, [((2, 2, 2), 64 * 513 + 1, 0.5, (0, 0, 0))], 500),
}


def run_case(ctx, name, theta, softening="spline", mass=False, seed=11):
    K, R, box, eps, cl, nbg = CASES[name]
    Gm = 1.0e-3
    pos = inputs.clumps(seed, K, box, cl, nbg)
    N = pos.shape[0]
    m = None
    if mass:
        m = (np.random.default_rng(seed + 1).random(N) + 0.5).astype(np.float32)
        b = ctx.bin(torch.from_numpy(pos).cuda(), K, box, mass=torch.from_numpy(m).cuda())
    else:
        b = ctx.bin(torch.from_numpy(pos).cuda(), K, box)
    amax = torch.zeros(K ** 3, dtype=torch.float32, device="cuda")
    acc = ctx.forces_tree(b, R, eps, Gm, theta, softening=softening, use_mass=mass, cell_amax=amax)
    st = ctx.tree_stats()
    acc = acc.cpu().numpy()
    assert np.isfinite(acc).all()
    return pos, m, b, acc, amax.cpu().numpy(), st, (K, R, box, eps, Gm)


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("theta", [0.5, 0.8])
def test_tree_matches_its_oracle(ctx, name, theta):
    pos, m, b, acc, amax, st, (K, R, box, eps, Gm) = run_case(ctx, name, theta)
    N = pos.shape[0]
    sinks = None if N <= 20000 else np.random.default_rng(3).choice(N, 6000, replace=False)
    ref, st_ref = nf_tree.forces_tree(pos, K, R, eps, box, Gm, theta, sink_idx=sinks, stats=True)
    assert st["node"] == st_ref["node"] and st["leaf"] == st_ref["leaf"]         # the same walk, bit for bit
    assert st["node"] > 0
    got = acc if sinks is None else acc[sinks]
    err = oracle.parity_error(got, ref)
    assert np.median(err) < MEDIAN_TOL and err.max() < MAX_TOL, (np.median(err), err.max())
    # per-cell maximum of |a| from the final accelerations
    key, _ = oracle.keys(pos, K, box)
    mag = np.sqrt((acc.astype(np.float32) ** 2).sum(axis=1, dtype=np.float32))
    want = np.zeros(K ** 3, dtype=np.float32)
    np.maximum.at(want, key, mag)
    assert np.allclose(amax, want, rtol=2e-6, atol=0)


@pytest.mark.parametrize("softening,mass", [("plummer", False), ("spline", True), ("plummer", True)])
def test_tree_variants(ctx, softening, mass):
    pos, m, b, acc, amax, st, (K, R, box, eps, Gm) = run_case(ctx, "three-clumps-R1", 0.6, softening=softening, mass=mass)
    ref, st_ref = nf_tree.forces_tree(pos, K, R, eps, box, Gm, 0.6, softening=softening, mass=m, stats=True)
    assert st["node"] == st_ref["node"] and st["leaf"] == st_ref["leaf"]
    err = oracle.parity_error(acc, ref)
    assert np.median(err) < MEDIAN_TOL and err.max() < MAX_TOL, (np.median(err), err.max())


def test_theta_zero_is_the_direct_sum(ctx):
    pos, m, b, acc, amax, st, (K, R, box, eps, Gm) = run_case(ctx, "two-clumps-R2-wrap", 0.0)
    assert st["node"] == 0
    direct = ctx.forces(b, R, eps, Gm).cpu().numpy()
    err = oracle.parity_error(acc, direct.astype(np.float64))
    assert err.max() < 2e-5
    ref = oracle.forces(pos, K, R, eps, box, Gm)
    err = oracle.parity_error(acc, ref)
    assert np.median(err) < MEDIAN_TOL and err.max() < MAX_TOL
    # every (sink, source of a dense neighbour cell) pair was met particle by particle
    cnt = b.cell_count.cpu().numpy().astype(np.int64).reshape(K, K, K)
    dense = nf_tree.dense_cells(cnt.ravel(), pos.shape[0]).reshape(K, K, K)
    tot = 0
    for d in np.ndindex(2 * R + 1, 2 * R + 1, 2 * R + 1):
        sh = np.roll(np.where(dense, cnt, 0), shift=(R - d[0], R - d[1], R - d[2]), axis=(0, 1, 2))
        tot += int((cnt * sh).sum())
    assert st["leaf"] == tot


def test_tree_is_reproducible_and_plain_without_dense_cells(ctx):
    pos, m, b, acc, amax, st, (K, R, box, eps, Gm) = run_case(ctx, "three-clumps-R1", 0.5)
    acc2 = ctx.forces_tree(b, R, eps, Gm, 0.5).cpu().numpy()
    assert np.array_equal(acc.view(np.uint32), acc2.view(np.uint32))
    # no dense cell: nothing for the tree to do, the direct sum
    rng = np.random.default_rng(5)
    for N in (3000, 30000):
        p2 = rng.random((N, 3)).astype(np.float32)
        b2 = ctx.bin(torch.from_numpy(p2).cuda(), 4, 1.0)
        a_t = ctx.forces_tree(b2, 1, 0.01, 1e-3, 0.7).cpu().numpy()
        assert ctx.tree_stats() == {"node": 0, "leaf": 0} or N < 4096
        a_d = ctx.forces(b2, 1, 0.01, 1e-3).cpu().numpy()
        assert oracle.parity_error(a_t, a_d.astype(np.float64)).max() < 2e-5


def test_tree_rejects_bad_theta(ctx):
    from paper_1810_02916_b200 import nf
    p2 = np.random.default_rng(6).random((5000, 3)).astype(np.float32)
    b2 = ctx.bin(torch.from_numpy(p2).cuda(), 3, 1.0)
    for th in (-0.1, 1.0, float("nan")):
        with pytest.raises(nf.NFError):
            ctx.forces_tree(b2, 1, 0.01, 1e-3, th)


@pytest.mark.parametrize("seed", [101, 102, 103, 104, 105])
def test_tree_randomised(ctx, seed):
    """Seeded random boxes: 1-3 clumps of 4096-9000 particles of random place, radius and offset, random K, R, eps, theta,
    softening law and masses.  Counts bit for bit, every sink within the bars."""
    rng = np.random.default_rng(seed)
    K = int(rng.integers(3, 7))
    R = 2 if (K >= 5 and rng.integers(0, 2)) else 1
    box = float(rng.choice([1.0, 3.0, 500.0]))
    w = box / K
    eps = float(w * rng.choice([0.002, 0.01, 0.05, 0.2]))
    theta = float(rng.choice([0.2, 0.4, 0.6, 0.8, 0.95]))
    cl = []
    for _ in range(int(rng.integers(1, 4))):
        rad = float(rng.choice([0.02, 0.1, 0.3, 0.49]))
        cl.append((tuple(int(x) for x in rng.integers(0, K, 3)), int(rng.choice([4096, 4100, 5000, 9000])), rad,
                   tuple(float(x) for x in rng.uniform(-0.4, 0.4, 3) * (0.5 - rad))))
    softening = str(rng.choice(["spline", "spline", "plummer"]))
    pos = inputs.clumps(seed, K, box, cl, int(rng.choice([0, 300, 3000])))
    N = pos.shape[0]
    m = (rng.random(N) + 0.5).astype(np.float32) if rng.integers(0, 2) else None
    b = ctx.bin(torch.from_numpy(pos).cuda(), K, box, mass=torch.from_numpy(m).cuda() if m is not None else None)
    acc = ctx.forces_tree(b, R, eps, 1e-3, theta, softening=softening, use_mass=m is not None).cpu().numpy()
    st = ctx.tree_stats()
    ref, st_ref = nf_tree.forces_tree(pos, K, R, eps, box, 1e-3, theta, softening=softening, mass=m, stats=True)
    assert st["node"] == st_ref["node"] and st["leaf"] == st_ref["leaf"]
    err = oracle.parity_error(acc, ref)
    assert np.isfinite(acc).all() and np.median(err) < MEDIAN_TOL and err.max() < MAX_TOL, (np.median(err), err.max())
