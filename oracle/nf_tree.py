"""CPU oracle of the TREE near field for dense cells -- plain numpy, double precision.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as nf_oracle.c: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import it; it shares no code with paper_1810_02916_b200/).

What the paper says: "Future versions of Abacus will employ trees in the near-field domain, especially for dense cells"
(PAPER.md:49); "the largest cell has over 200,000 particles".  It prints no algorithm, so this file follows
the one DESIGN.md states (readings t1-t6, "Tree near field"), step by step:

  t1  A cell is DENSE when it holds >= 4096 particles.  (Capacity rule of the implementation, part of the definition: the
      dense cells taken are, in cell order, the first 2048 whose 64-aligned sizes add up to at most
      cap(N) = min(max(N, 2^20) + 64 * 2048, 2^28) rounded down to 64 -- room for every particle unless N > 2^28 --; further
      ones are treated as not dense.)
  t2  Inside a dense cell the particles are ordered by the 21-bit Hilbert index (Skilling's construction) of their float32
      cell-centred offset o (7 bits per axis, q = clamp(int(((o * (K/box)) + 0.5) * 128), 0, 127), every operation
      rounded to float32, x the most significant axis), ties in the stable order of the binning.  (A Hilbert run is a
      compact blob; a Morton run jumps across the cell at octant boundaries and its bounding box with it.)
  t3  LEAVES are runs of 16 consecutive particles of that order; a node of level l holds 8 consecutive nodes of level
      l-1, up to a single root.  A node carries the bounding box of its particles' float32 offsets, its mass M and its
      centre of mass.
  t4  SINK GROUPS are runs of 64 consecutive particles of a cell, in Hilbert order if the cell is dense and in the binned
      order if not; a group carries the bounding box of its float32 offsets.  A group whose box is more than 3 times
      larger (diagonal) than the smallest box of its four quarters walks quarter by quarter, and a quarter that is
      itself that large walks sink by sink (group_parts): one outlier must not make a whole group open the whole tree.
  t5  A group meets a dense cell at cell displacement delta (|delta| <= R per axis, periodic) by walking its tree from
      the root.  With sh = float32(delta) * float32(box/K), a node box shifted by sh, g = the per-axis gap between the two
      boxes (0 when they overlap), d2 = (gx*gx + gy*gy) + gz*gz, s2 = (ex*ex + ey*ey) + ez*ez for the node's extents e
      -- all float32, no fused multiply-add -- the node is ACCEPTED when d2 > eps^2 and s2 < theta^2 * d2.  An accepted
      node acts on every sink of the group as one particle of mass M at its centre of mass (1/r^2 law: every replaced pair
      is further apart than eps); a node that is not accepted is opened (its children are tested), and a leaf that is not
      accepted is summed particle by particle with the full softened law.
  t6  Sources in cells that are not dense act by the direct sum of PAPER.md:37, unchanged.

theta = 0 accepts nothing and IS the direct sum.  For theta > 0 the result is an approximation with the classical
monopole bound: for a sink at distance D from the centre of mass of a node whose particles lie within b < theta * D of it,
|error| <= G M / D^2 * (1/(1-theta)^2 - 1 - 2 theta).

The float32 decisions (t2, t5) are taken in the same precision by the CUDA path, so the two walks are the same walk;
everything else here is double precision from the caller's float32 positions, as in nf_oracle.c.

Pins (tests/test_tree_oracle_pins.py): theta = 0 equals nf_oracle.forces; a far, tight dense cell seen from a single sink
equals the hand formula G M (c - x)/|c - x|^3; the error against the direct sum respects the bound above sink by sink and
falls with theta; conservation of the interaction count at theta = 0 (every sink meets every source of a dense neighbour).
"""
from __future__ import annotations

import itertools

import numpy as np

from . import nf_oracle as _o

LEAF = 16
GROUP = 64
FANOUT = 8
DENSE_N = 4096
DENSE_MAX_CELLS = 2048
f32 = np.float32


def dense_cap(N: int) -> int:
    c = max(N, 1 << 20) + 64 * DENSE_MAX_CELLS
    return min(c, 1 << 28) & ~63


def dense_cells(cell_count, N: int):
    """t1: boolean mask of the dense cells taken."""
    cnt = np.asarray(cell_count, dtype=np.int64)
    big = cnt >= DENSE_N
    n64 = np.where(big, (cnt + 63) & ~63, 0)
    coff = np.cumsum(n64) - n64
    rank = np.cumsum(big) - big
    return big & (rank < DENSE_MAX_CELLS) & (coff + n64 <= dense_cap(int(N)))


def hilbert_index(q, bits: int = 7):
    """Hilbert index of integer grid points q [n, 3] (J. Skilling, "Programming the Hilbert curve", AIP Conf. Proc. 707,
    2004: the transpose construction), axis 0 the most significant.  Consecutive indices are face-adjacent cells."""
    X = [np.array(q[:, a], dtype=np.uint32) for a in range(3)]
    Q = 1 << (bits - 1)
    while Q > 1:
        P = np.uint32(Q - 1)
        for i in range(3):
            hit = (X[i] & np.uint32(Q)) != 0
            t = (X[0] ^ X[i]) & P
            x0 = np.where(hit, X[0] ^ P, X[0] ^ t)       # invert the low bits of X[0] / exchange them with X[i]'s
            xi = np.where(hit, X[i], X[i] ^ t)
            X[i] = xi
            X[0] = x0
        Q >>= 1
    X[1] = X[1] ^ X[0]                                   # Gray encode
    X[2] = X[2] ^ X[1]
    t = np.zeros_like(X[0])
    Q = 1 << (bits - 1)
    while Q > 1:
        t = np.where((X[2] & np.uint32(Q)) != 0, t ^ np.uint32(Q - 1), t)
        Q >>= 1
    h = np.zeros_like(X[0])
    for b in range(bits):
        for a in range(3):
            h |= (((X[a] ^ t) >> b) & 1) << (3 * b + (2 - a))
    return h


def hilbert_order(off32, K: int, box: float):
    """t2: the in-cell order (indices into the cell's particles in binned order)."""
    invw = f32(K) / f32(box)
    o = np.asarray(off32, dtype=f32)
    t = ((o * invw).astype(f32) + f32(0.5)).astype(f32)
    q = np.clip((t * f32(128.0)).astype(f32).astype(np.int32), 0, 127).astype(np.uint32)
    return np.argsort(hilbert_index(q, 7), kind="stable")


def build_tree(off32, xg, m):
    """t3: levels[0] = leaves ... levels[-1] = root; each a dict of lo, hi (float32 [n,3]), mass, com (float64).
    off32, xg (double global positions), m (double masses) are in Hilbert order."""
    n = off32.shape[0]
    nl = (n + LEAF - 1) // LEAF
    lo = np.empty((nl, 3), dtype=f32)
    hi = np.empty((nl, 3), dtype=f32)
    mass = np.empty(nl)
    mx = np.empty((nl, 3))
    for k in range(nl):
        s = slice(k * LEAF, min(n, (k + 1) * LEAF))
        lo[k] = off32[s].min(axis=0)
        hi[k] = off32[s].max(axis=0)
        mass[k] = m[s].sum()
        mx[k] = (m[s, None] * xg[s]).sum(axis=0)
    levels = [dict(lo=lo, hi=hi, mass=mass, mx=mx)]
    while levels[-1]["mass"].shape[0] > 1:
        p = levels[-1]
        nn = (p["mass"].shape[0] + FANOUT - 1) // FANOUT
        lo = np.empty((nn, 3), dtype=f32)
        hi = np.empty((nn, 3), dtype=f32)
        mass = np.empty(nn)
        mx = np.empty((nn, 3))
        for k in range(nn):
            s = slice(k * FANOUT, (k + 1) * FANOUT)
            lo[k] = p["lo"][s].min(axis=0)
            hi[k] = p["hi"][s].max(axis=0)
            mass[k] = p["mass"][s].sum()
            mx[k] = p["mx"][s].sum(axis=0)
        levels.append(dict(lo=lo, hi=hi, mass=mass, mx=mx))
    for L in levels:
        # a node of zero mass (massless particles only) never attracts; its centre is irrelevant
        L["com"] = L["mx"] / np.where(L["mass"] != 0, L["mass"], 1.0)[:, None]
    return levels


def accept(glo, ghi, nlo, nhi, sh, eps, theta):
    """t5: the opening criterion, float32, for arrays of node boxes."""
    nlo_s = (nlo + sh).astype(f32)
    nhi_s = (nhi + sh).astype(f32)
    g = np.maximum(np.maximum((glo - nhi_s).astype(f32), (nlo_s - ghi).astype(f32)), f32(0.0))
    gg = (g * g).astype(f32)
    d2 = ((gg[:, 0] + gg[:, 1]).astype(f32) + gg[:, 2]).astype(f32)
    e = (nhi - nlo).astype(f32)
    ee = (e * e).astype(f32)
    s2 = ((ee[:, 0] + ee[:, 1]).astype(f32) + ee[:, 2]).astype(f32)
    eps2 = f32(f32(eps) * f32(eps))
    th2 = f32(f32(theta) * f32(theta))
    return (d2 > eps2) & (s2 < (th2 * d2).astype(f32))


def walk(levels, glo, ghi, sh, eps, theta):
    """t5: (list of (level, node) accepted, array of leaves to be summed directly)."""
    acc_nodes = []
    top = len(levels) - 1
    front = np.array([0], dtype=np.int64)
    for l in range(top, -1, -1):
        L = levels[l]
        ok = accept(glo, ghi, L["lo"][front], L["hi"][front], sh, eps, theta)
        for k in front[ok]:
            acc_nodes.append((l, int(k)))
        opened = front[~ok]
        if l == 0:
            return acc_nodes, opened
        nchild = levels[l - 1]["mass"].shape[0]
        ch = (opened[:, None] * FANOUT + np.arange(FANOUT)[None, :]).ravel()
        front = ch[ch < nchild]
    raise AssertionError


def _diag2(lo, hi):
    e = (hi - lo).astype(f32)
    ee = (e * e).astype(f32)
    return f32(f32(ee[0] + ee[1]) + ee[2])


def group_parts(o32, theta: float = 1.0):
    """t4: how the (up to 64) sinks of a group walk -- a list of (box lo, box hi, member positions).  Normally all
    together under the box of the group.  A group whose box is out of proportion (an outlier among its sinks makes every
    node look close, and the walk opens the whole tree) walks in parts: with m = the smallest squared diagonal among the
    boxes of its four quarters (16 consecutive sinks each; quarters of fewer than 8 sinks do not count, and with none
    that counts the group is not split), the group is split when its own squared diagonal exceeds 9 m; then each quarter walks under its own box, except that a quarter whose squared diagonal
    exceeds 9 m walks sink by sink (a point has no extent).  float32, every operation rounded.  With theta = 0 nothing
    is ever accepted, no box is looked at, and the group walks as a whole."""
    n = o32.shape[0]
    lo, hi = o32.min(axis=0), o32.max(axis=0)
    if f32(f32(theta) * f32(theta)) == 0:
        return [(lo, hi, np.arange(n))]
    quarters = [np.arange(16 * q, min(n, 16 * q + 16)) for q in range(4) if 16 * q < n]
    d2q = [_diag2(o32[m].min(axis=0), o32[m].max(axis=0)) for m in quarters]
    counted = [d2 for m, d2 in zip(quarters, d2q) if m.shape[0] >= 8]
    if not counted:
        return [(lo, hi, np.arange(n))]
    lim = f32(f32(9.0) * min(counted))
    if not _diag2(lo, hi) > lim:
        return [(lo, hi, np.arange(n))]
    parts = []
    for m, d2 in zip(quarters, d2q):
        if d2 > lim:
            parts += [(o32[i], o32[i], np.array([i])) for i in m]
        else:
            parts.append((o32[m].min(axis=0), o32[m].max(axis=0), m))
    return parts


def _law(d, eps, softening):
    """|F|/r for displacement vectors d [.., 3]; r = 0 contributes nothing (reading c6)."""
    r2 = (d * d).sum(axis=-1)
    if softening == "plummer":
        s = r2 + eps * eps
        return 1.0 / (s * np.sqrt(s))
    r = np.sqrt(r2)
    u = r / eps
    with np.errstate(divide="ignore", invalid="ignore"):
        far = np.where(r2 > 0, 1.0 / (r2 * r), 0.0)
    return np.where(u < 1.0, (10.0 - 15.0 * u + 6.0 * u * u) / eps ** 3, far)


def forces_tree(pos, K: int, R: int, eps: float, box: float, Gm: float, theta: float, softening: str = "spline",
                mass=None, sink_idx=None, stats: bool = False):
    """Near-field accelerations with the tree for dense source cells (t1-t6).  float64 [n_sinks, 3] in the order of
    sink_idx (all particles, input order, if None).  stats=True also returns a dict of interaction counts:
    node = sum over (sink, accepted node) pairs, leaf = sum over (sink, particle of an opened leaf) pairs,
    direct = ordered pairs whose source cell is not dense."""
    pos = np.ascontiguousarray(pos, dtype=f32)
    N = pos.shape[0]
    b = _o.bin_particles(pos, K, box)
    cnt = b["cell_count"].astype(np.int64)
    off = b["cell_offset"].astype(np.int64)
    perm = b["perm"].astype(np.int64)
    offs32 = b["pos_sorted"][:, :3]
    dense = dense_cells(cnt, N)
    key, _ = _o.keys(pos, K, box)
    m_all = np.ones(N) if mass is None else np.asarray(mass, dtype=f32).astype(np.float64)
    # t6: the direct sum over sources of cells that are not dense (their masses kept, the others' set to zero)
    m_direct = np.where(dense[key], 0.0, m_all).astype(f32)
    want = np.arange(N) if sink_idx is None else np.asarray(sink_idx, dtype=np.int64)
    a = _o.forces(pos, K, R, eps, box, Gm, sink_idx=want, softening=softening, mass=m_direct)
    wanted = np.zeros(N, dtype=bool)
    wanted[want] = True
    a_tree = np.zeros((N, 3))
    xg = pos.astype(np.float64)
    st = dict(node=0, leaf=0, direct=0)
    # trees of the dense cells, built when first needed
    trees = {}

    def tree_of(c):
        if c not in trees:
            s = np.arange(off[c], off[c + 1])
            s = s[hilbert_order(offs32[s], K, box)]
            trees[c] = (s, build_tree(offs32[s], xg[perm[s]], m_all[perm[s]]))
        return trees[c]

    cw32 = f32(box) / f32(K)
    deltas = list(itertools.product(range(-R, R + 1), repeat=3))
    cells = np.nonzero(cnt > 0)[0]
    for c in cells:
        if not stats and not wanted[perm[off[c]:off[c + 1]]].any():
            continue
        cz, cy, cx = int(c % K), int((c // K) % K), int(c // (K * K))
        nb = []
        for (dx, dy, dz) in deltas:
            qx, qy, qz = cx + dx, cy + dy, cz + dz
            D = ((qx % K) * K + (qy % K)) * K + (qz % K)
            if dense[D]:
                nb.append((D, (dx, dy, dz), (qx // K, qy // K, qz // K)))
            elif stats:
                st["direct"] += int(cnt[c]) * int(cnt[D])
        if not nb:
            continue
        s_c = tree_of(int(c))[0] if dense[c] else np.arange(off[c], off[c + 1])
        for g0 in range(0, s_c.shape[0], GROUP):
            gs = s_c[g0:g0 + GROUP]                      # t4: sorted slots of the group's sinks
            if not stats and not wanted[perm[gs]].any():
                continue
            for (glo, ghi, members) in group_parts(offs32[gs], theta):
                ps = gs[members]                         # t4: the sinks that walk together, and their box
                xs = xg[perm[ps]]
                for (D, dl, img) in nb:
                    src, levels = tree_of(int(D))
                    sh = (np.array(dl, dtype=f32) * cw32).astype(f32)
                    nodes, leaves = walk(levels, glo, ghi, sh, eps, theta)
                    image = np.array(img, dtype=np.float64) * float(box)
                    if nodes:
                        com = np.array([levels[l]["com"][k] for (l, k) in nodes]) + image
                        M = np.array([levels[l]["mass"][k] for (l, k) in nodes])
                        d = com[None, :, :] - xs[:, None, :]
                        r2 = (d * d).sum(axis=-1)
                        if softening == "plummer":
                            fr = _law(d, eps, softening)
                        else:
                            fr = 1.0 / (r2 * np.sqrt(r2))
                        a_tree[perm[ps]] += Gm * ((M[None, :] * fr)[:, :, None] * d).sum(axis=1)
                        st["node"] += len(nodes) * ps.shape[0]
                    if leaves.size:
                        idx = np.concatenate([src[k * LEAF:(k + 1) * LEAF] for k in leaves])
                        d = (xg[perm[idx]] + image)[None, :, :] - xs[:, None, :]
                        fr = _law(d, eps, softening)
                        a_tree[perm[ps]] += Gm * ((m_all[perm[idx]][None, :] * fr)[:, :, None] * d).sum(axis=1)
                        st["leaf"] += idx.shape[0] * ps.shape[0]
    out = a + a_tree[want]
    return (out, st) if stats else out


def monopole_bound(theta: float) -> float:
    """sum_{k>=2} (k+1) theta^k: relative bound of the monopole error of one accepted node (header)."""
    return 1.0 / (1.0 - theta) ** 2 - 1.0 - 2.0 * theta
