"""Pins for the tree near field oracle (oracle/nf_tree.py, readings t1-t6).  Every check compares it
with something other than itself: the direct-sum oracle (itself pinned by test_oracle_pins.py), a hand formula, the
classical monopole error bound, geometric invariants of the Hilbert order and of the boxes."""
import numpy as np

import oracle
from oracle import nf_tree
from paper_1810_02916_b200 import inputs


def clumpy(seed, K, box, clumps, n_bg):
    return inputs.clumps(seed, K, box, clumps, n_bg)


def test_theta_zero_is_the_direct_sum_and_counts_every_pair():
    K, R, box, eps, Gm = 4, 1, 4.0, 0.02, 1.0e-3
    pos = clumpy(1, K, box, [((1, 1, 1), 4500, 0.3, (0.1, 0, 0)), ((1, 1, 2), 4200, 0.45, (0, 0, -0.05)),
                            ((3, 0, 1), 4100, 0.2, (0, 0.2, 0))], 1500)
    sinks = np.random.default_rng(2).choice(pos.shape[0], 600, replace=False)
    for soft in ("spline", "plummer"):
        a_dir = oracle.forces(pos, K, R, eps, box, Gm, sink_idx=sinks, softening=soft)
        a_tree = nf_tree.forces_tree(pos, K, R, eps, box, Gm, 0.0, softening=soft, sink_idx=sinks)
        scale = np.abs(a_dir).max()
        assert np.abs(a_tree - a_dir).max() <= 1e-12 * scale
    _, st = nf_tree.forces_tree(pos, K, R, eps, box, Gm, 0.0, stats=True)
    b = oracle.bin_particles(pos, K, box)
    assert st["node"] == 0
    assert st["leaf"] + st["direct"] == oracle.interactions(b["cell_count"], K, R)
    assert nf_tree.dense_cells(b["cell_count"], pos.shape[0]).sum() == 3


def test_far_tight_dense_cell_is_a_point_mass_hand_formula():
    """One dense cell holding a tight ball, single sinks two cells away (one of them through the periodic wrap):
    with theta = 0.5 the root is accepted and the acceleration is G M (c - x)/|c - x|^3 by hand."""
    K, R, box, eps, Gm = 5, 2, 5.0, 0.2, 2.5e-4          # eps wider than the ball: no node can be accepted inside it
    rng = np.random.default_rng(3)
    ball = (np.array([2.5, 2.5, 0.5]) + 0.01 * rng.normal(size=(4096, 3))).astype(np.float32)
    s1 = np.array([[4.3, 2.4, 0.6]], dtype=np.float32)      # delta = (-2, 0, 0), no wrap
    s2 = np.array([[2.6, 2.5, 3.4]], dtype=np.float32)      # cell z = 3: delta z = +2 wraps to cell 0, image +box
    pos = np.concatenate([ball, s1, s2])
    a, st = nf_tree.forces_tree(pos, K, R, eps, box, Gm, 0.5, stats=True)
    com = ball.astype(np.float64).mean(axis=0)
    # the two single sinks also see each other (cells (4,2,0) and (2,2,3): delta z = -2 / +2 through the wrap), directly
    d12 = s2[0].astype(np.float64) - s1[0].astype(np.float64) - np.array([0, 0, box])
    for i, x, image, pair in ((4096, s1[0], (0, 0, 0), d12), (4097, s2[0], (0, 0, box), -d12)):
        d = com + np.array(image, dtype=np.float64) - x.astype(np.float64)
        hand = Gm * 4096 * d / np.linalg.norm(d) ** 3 + Gm * pair / np.linalg.norm(pair) ** 3
        assert np.abs(a[i] - hand).max() <= 1e-12 * np.abs(hand).max()
    # the two single sinks each met one node (the root); inside the ball every pair was summed
    assert st["node"] == 2 and st["leaf"] == 4096 * 4096
    # and the monopole differs from the direct sum by the quadrupole of a 0.01-ball at distance ~1.8: ~ (0.02/1.8)^2
    a_dir = oracle.forces(pos, K, R, eps, box, Gm, sink_idx=np.array([4096, 4097]))
    rel = np.abs(a[4096:] - a_dir).max() / np.abs(a_dir).max()
    assert 0 < rel < 5e-4


def test_error_bound_sink_by_sink_and_convergence():
    K, R, box, eps, Gm = 4, 1, 4.0, 0.01, 1.0
    pos = clumpy(5, K, box, [((2, 2, 2), 6000, 0.5, (0, 0, 0)), ((2, 2, 3), 4300, 0.35, (0.1, -0.1, 0))], 800)
    N = pos.shape[0]
    sinks = np.random.default_rng(6).choice(N, 400, replace=False)
    a_dir = oracle.forces(pos, K, R, eps, box, Gm, sink_idx=sinks)
    # S_i = sum of G m / r^2 over the sources of dense neighbour cells further than eps, by brute force in numpy
    b = oracle.bin_particles(pos, K, box)
    key, _ = oracle.keys(pos, K, box)
    dense = nf_tree.dense_cells(b["cell_count"], N)
    src = np.nonzero(dense[key])[0]
    x = pos.astype(np.float64)
    rms = []
    for theta in (0.7, 0.35):
        a_t, st = nf_tree.forces_tree(pos, K, R, eps, box, Gm, theta, sink_idx=sinks), None
        err = np.linalg.norm(a_t - a_dir, axis=1)
        bound = np.empty(sinks.shape[0])
        for n, i in enumerate(sinks):
            d = x[src] - x[i]
            d -= box * np.round(d / box)
            r2 = (d * d).sum(axis=1)
            bound[n] = Gm * (1.0 / r2[r2 > eps * eps]).sum()
        bound *= nf_tree.monopole_bound(theta) * (1 + theta) ** 2
        assert (err <= bound).all()
        rms.append(np.sqrt((err ** 2).mean()))
    assert rms[0] > 0 and rms[1] < 0.5 * rms[0]           # it does approximate, and the error falls with theta
    mag = np.linalg.norm(a_dir, axis=1)
    assert rms[1] / np.sqrt((mag ** 2).mean()) < 5e-3


def test_hilbert_index_brute_force():
    """Every point of the 16^3 grid gets its own index and consecutive indices are face-adjacent cells -- the defining
    property of the curve, checked exhaustively; x is the most significant axis (the curve ends at (15, 0, 0))."""
    n = 16
    g = np.stack(np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij"), -1).reshape(-1, 3).astype(np.uint32)
    h = nf_tree.hilbert_index(g, 4)
    assert sorted(h.tolist()) == list(range(n ** 3))
    path = g[np.argsort(h)].astype(int)
    assert (np.abs(np.diff(path, axis=0)).sum(axis=1) == 1).all()
    assert path[0].tolist() == [0, 0, 0] and path[-1].tolist() == [n - 1, 0, 0]
    # the 7-bit curve used by the tree: a sample of consecutive indices, found by inverting on the full grid of one octant pair
    g7 = np.stack(np.meshgrid(np.arange(128), np.arange(64, 72), np.arange(128), indexing="ij"), -1).reshape(-1, 3).astype(np.uint32)
    h7 = nf_tree.hilbert_index(g7, 7)
    o = np.argsort(h7)
    hs, ps = h7[o].astype(np.int64), g7[o].astype(int)
    adj = np.diff(hs) == 1
    assert adj.sum() > 10000 and (np.abs(np.diff(ps, axis=0)).sum(axis=1)[adj] == 1).all()


def test_hilbert_order_and_boxes_invariants():
    K, box = 3, 3.0
    rng = np.random.default_rng(7)
    off = ((rng.random((5000, 3)) - 0.5) * (box / K) * 0.999).astype(np.float32)
    order = nf_tree.hilbert_order(off, K, box)
    assert sorted(order.tolist()) == list(range(5000))
    o = off[order]
    # each of the eight octants of the cell is one contiguous run along the curve, and so is each of the 64 sub-octants
    w = box / K
    for parts in (2, 4):
        sub = np.floor((o / w + 0.5) * parts).astype(int)
        ident = (sub[:, 0] * parts + sub[:, 1]) * parts + sub[:, 2]
        assert (np.diff(ident) != 0).sum() + 1 == parts ** 3
    # the curve starts in the octant of the low corner and ends across the cell in x
    assert (o[0] < 0).all() and o[-1, 0] > 0 and (o[-1, 1:] < 0).all()
    m = rng.random(5000) + 0.5
    xg = o.astype(np.float64) + 1.5
    levels = nf_tree.build_tree(o, xg, m)
    assert [L["mass"].shape[0] for L in levels] == [313, 40, 5, 1]
    assert abs(levels[-1]["mass"][0] - m.sum()) < 1e-9
    assert np.allclose(levels[-1]["com"][0], (m[:, None] * xg).sum(axis=0) / m.sum(), rtol=0, atol=1e-12)
    assert (levels[-1]["lo"][0] == o.min(axis=0)).all() and (levels[-1]["hi"][0] == o.max(axis=0)).all()
    for l in range(1, len(levels)):
        for k in range(levels[l]["mass"].shape[0]):
            ch = slice(8 * k, 8 * k + 8)
            assert (levels[l]["lo"][k] <= levels[l - 1]["lo"][ch]).all() and (levels[l]["hi"][k] >= levels[l - 1]["hi"][ch]).all()
    # a leaf's box is the box of ITS 16 particles
    assert (levels[0]["lo"][3] == o[48:64].min(axis=0)).all() and (levels[0]["hi"][312] == o[312 * 16:].max(axis=0)).all()


def test_opening_criterion_by_hand():
    f = np.float32
    glo, ghi = np.array([0, 0, 0], dtype=f), np.array([1, 1, 1], dtype=f)
    nlo = np.array([[3, 0, 0], [3, 0, 0], [1.5, 0, 0], [0.5, 0.5, 0.5]], dtype=f)
    nhi = np.array([[4, 1, 1], [5, 2, 2], [1.6, 0.1, 0.1], [0.6, 0.6, 0.6]], dtype=f)
    sh = np.zeros(3, dtype=f)
    # gaps 2, 2, 0.5, 0 (overlap); sizes^2 3, 12, 0.03, 0.03
    assert nf_tree.accept(glo, ghi, nlo, nhi, sh, 0.1, 1.0).tolist() == [True, False, True, False]
    assert nf_tree.accept(glo, ghi, nlo, nhi, sh, 0.1, 0.5).tolist() == [False, False, True, False]
    assert nf_tree.accept(glo, ghi, nlo, nhi, sh, 0.6, 1.0).tolist() == [True, False, False, False]     # inside eps: never
    assert nf_tree.accept(glo, ghi, nlo, nhi, sh, 0.1, 0.0).tolist() == [False] * 4
    # the shift moves the node: the third box shifted by +2 in x is at gap 2.5
    assert nf_tree.accept(glo, ghi, nlo[2:3], nhi[2:3], np.array([2, 0, 0], dtype=f), 2.4, 1.0).tolist() == [True]
    assert nf_tree.accept(glo, ghi, nlo[2:3], nhi[2:3], np.array([2, 0, 0], dtype=f), 2.6, 1.0).tolist() == [False]
    assert nf_tree.accept(glo, ghi, nlo[2:3], nhi[2:3], np.array([-3, 0, 0], dtype=f), 1.3, 1.0).tolist() == [True]   # gap 1.4 on the other side


def test_group_parts_by_hand():
    f = np.float32
    line = np.zeros((64, 3), dtype=f)
    line[:, 0] = np.arange(64)
    # a 4 x 4 x 4 lattice whose quarters are 4 x 4 x 1 slabs: group diagonal^2 = 27, quarters 18 -> walks as a whole
    cube = np.array([[i % 4, (i // 4) % 4, i // 16] for i in range(64)], dtype=f)
    p = nf_tree.group_parts(cube)
    assert len(p) == 1 and p[0][2].tolist() == list(range(64)) and p[0][0].tolist() == [0, 0, 0] and p[0][1].tolist() == [3, 3, 3]
    # a line of 64: extent 63 against 15 per quarter (63^2 > 9 * 15^2) -> four quarters, each under its own box
    p = nf_tree.group_parts(line)
    assert [(a[0], b[0], m.tolist()) for a, b, m in p] == [(16 * q, 16 * q + 15, list(range(16 * q, 16 * q + 16))) for q in range(4)]
    # one outlier in the second quarter: that quarter walks sink by sink (point boxes), the others as quarters
    out = line.copy()
    out[20] = [1000, 0, 0]
    p = nf_tree.group_parts(out)
    assert [m.tolist() for _, _, m in p] == [list(range(16))] + [[i] for i in range(16, 32)] + [list(range(32, 48)), list(range(48, 64))]
    assert all((a == b).all() and (a == out[m[0]]).all() for a, b, m in p[1:17])
    assert sorted(i for _, _, m in p for i in m.tolist()) == list(range(64))
    # a short group: the quarter of 4 sinks does not count (limit 9 * 15^2 = 2025 >= 19^2): as a whole; 7 sinks: nothing counts
    assert len(nf_tree.group_parts(line[:20])) == 1 and len(nf_tree.group_parts(line[:7])) == 1
    # ... but 24 sinks with the last 8 far away: the second quarter counts (8 sinks, extent 7) and the group splits
    far = line[:24].copy()
    far[16:, 0] += 500
    p = nf_tree.group_parts(far)
    assert [m.tolist() for _, _, m in p] == [list(range(16)), list(range(16, 24))]       # 15^2 <= 9 * 7^2: both stay quarters
