"""Pins for the CPU oracle (oracle/nf_oracle.c): every check here compares the oracle with
something OTHER than itself -- the paper's closed forms, brute force that shares no cell-list
code with it, invariants of the mathematics.  A plausible mistake in the oracle (dropped term,
wrong sign or index, wrong image, transposed axis) fails at least one of them.
"""
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- helpers
def cells_f32(pos, K, box):
    """Float32 cell index (the definitional contract) retyped in numpy."""
    invw = np.float32(K) / np.float32(box)
    c = np.floor(pos.astype(np.float32) * invw).astype(np.int64)
    return np.clip(c, 0, K - 1)


def brute_force(pos, K, R, eps, box, Gm, softening="spline"):
    """Pair-centric O(N^2) near-field sum (SURVEY.md Sec. 8(c) 'Pair set / periodic wrap'):
    for every ordered pair find per axis the unique delta in [-R, R] with
    (c_i + delta) mod K == c_j; otherwise the pair is not in the near field.  No cell lists."""
    x = pos.astype(np.float64)
    c = cells_f32(pos, K, box)
    n = x.shape[0]
    acc = np.zeros((n, 3))
    diff = (c[None, :, :] - c[:, None, :]) % K            # [i, j, axis]
    delta = np.where(diff <= R, diff, np.where(diff >= K - R, diff - K, 10 ** 6))
    near = (np.abs(delta) <= R).all(axis=2)
    img = (c[:, None, :] + delta - c[None, :, :]) // K      # image shift n in {-1,0,1}
    for i in range(n):
        js = np.nonzero(near[i])[0]
        d = x[js] + img[i, js] * float(box) - x[i]
        r2 = (d * d).sum(axis=1)
        ok = r2 > 0
        d, r = d[ok], np.sqrt(r2[ok])
        if softening == "spline":
            u = r / eps
            f = np.where(u < 1, (10 - 15 * u + 6 * u * u) / eps ** 3, 1.0 / r ** 3)
        else:
            f = (r * r + eps * eps) ** -1.5
        acc[i] = Gm * (f[:, None] * d).sum(axis=0)
    return acc


def read_golden(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as fh:
        for line in fh:
            line = line.split("#")[0].strip()
            if line:
                rows.append([float(t) for t in line.split()])
    return np.array(rows)


# ----------------------------------------------------------------------------- Eq. 2 itself
def test_spline_coefficients_from_c2_conditions():
    """'requiring a smooth transition at the softening scale up to the second
    derivative'.  With F/r = s(u)/eps^3, s = a + b u + c u^2 must match u^-3 in value, first
    and second derivative at u = 1: s(1)=1, s'(1)=-3, s''(1)=12.  Unique solution (10,-15,6)."""
    M = np.array([[1, 1, 1], [0, 1, 2], [0, 0, 2]], dtype=float)
    a, b, c = np.linalg.solve(M, np.array([1.0, -3.0, 12.0]))
    assert np.allclose([a, b, c], [10, -15, 6])
    eps = 0.37
    for u in np.linspace(0.01, 0.99, 23):
        assert oracle.spline_over_r(u * eps, eps) == pytest.approx((a + b * u + c * u * u) / eps ** 3, rel=1e-14)


def test_spline_c2_continuity_at_eps():
    """Value, first and second derivative of F/r are continuous at r = eps (numerical)."""
    eps = 0.125
    h = 1e-4 * eps
    f = lambda r: oracle.spline_over_r(r, eps)
    # one-sided finite differences from each side
    left = [f(eps - k * h) for k in range(0, 4)]
    right = [f(eps + k * h) for k in range(0, 4)]
    d1l = (left[0] - left[1]) / h
    d1r = (right[1] - right[0]) / h
    d2l = (left[0] - 2 * left[1] + left[2]) / h ** 2
    d2r = (right[0] - 2 * right[1] + right[2]) / h ** 2
    assert left[0] == pytest.approx(1 / eps ** 3, rel=1e-14)
    assert d1l == pytest.approx(d1r, rel=2e-3)
    assert d2l == pytest.approx(d2r, rel=2e-2)
    assert d1l == pytest.approx(-3 / eps ** 4, rel=2e-3)
    assert d2l == pytest.approx(12 / eps ** 5, rel=2e-2)


def test_min_identity_footnote4():
    """PAPER.md:239 (fn. 4): the split is 'a single min'.  p(u) = 6u^5-15u^4+10u^3-1 is monotone
    with its only root at u=1, so min(s(u), u^-3)/eps^3 is Eq. 2 for every u>0."""
    eps = 0.8
    for u in np.concatenate([np.linspace(0.05, 0.999, 40), np.linspace(1.0, 6.0, 40)]):
        s = 10 - 15 * u + 6 * u * u
        assert oracle.spline_over_r(u * eps, eps) == pytest.approx(min(s, u ** -3) / eps ** 3, rel=1e-13)
    assert 1.36 < 0.9 ** -3 and 0.76 > 1.1 ** -3 and 0.625 > 1.25 ** -3     # the fixture's spot values


def test_spline_plummer_equivalence_factor():
    """eps_s = 2.16 eps_p gives the same minimum pairwise dynamical time.  The
    orbital frequency^2 for a pair is F/r, maximal at r -> 0: 10/eps_s^3 (Eq. 2) vs 1/eps_p^3
    (Eq. 1), equal for eps_s = 10^(1/3) eps_p = 2.154 eps_p ~ 2.16."""
    assert abs(10 ** (1 / 3) - 2.16) < 0.01
    eps_p = 0.3
    eps_s = 10 ** (1 / 3) * eps_p
    assert oracle.spline_over_r(1e-9, eps_s) == pytest.approx(oracle.plummer_over_r(1e-9, eps_p), rel=1e-6)


# ----------------------------------------------------------------------------- two particles
@pytest.mark.parametrize("placement", ["same_cell", "across_face", "across_box_edge", "diagonal"])
def test_two_particle_closed_form(placement):
    """Golden values of tests/golden/spline_closed_form.txt (Eq. 2 by hand), through the full
    oracle path (binning, neighbour cells, periodic image, direction and sign)."""
    gold = read_golden("spline_closed_form.txt")
    K, R, box, Gm = 8, 2, 1.0, 0.75
    w = box / K
    eps = w / 16                     # power of two so that positions are exact in float32
    for u, expect in gold:
        r = u * eps
        if placement == "same_cell":
            p0 = np.array([3.5 * w, 2.5 * w, 4.5 * w]); dirn = np.array([1.0, 0.0, 0.0])
        elif placement == "across_face":
            p0 = np.array([3.0 * w - r / 2, 2.5 * w, 4.5 * w]); dirn = np.array([1.0, 0.0, 0.0])
        elif placement == "across_box_edge":
            p0 = np.array([1.5 * w, box - r / 2, 0.5 * w]); dirn = np.array([0.0, 1.0, 0.0])
        else:
            p0 = np.array([3.5 * w, 2.5 * w, 4.5 * w]); dirn = np.array([2.0, -1.0, 2.0]) / 3.0
        p1 = p0 + r * dirn
        pos = np.mod(np.stack([p0, p1]), box).astype(np.float32)
        # the float32 rounding of the positions changes r slightly: use the realised separation
        d = pos[1].astype(np.float64) - pos[0].astype(np.float64)
        d -= np.round(d / box) * box
        ureal = np.linalg.norm(d) / eps
        expect_real = ureal * (10 - 15 * ureal + 6 * ureal ** 2) if ureal < 1 else ureal ** -2
        assert expect_real == pytest.approx(expect, rel=1e-4)        # the fixture value itself
        a = oracle.forces(pos, K, R, eps, box, Gm)
        assert np.linalg.norm(a[0]) * eps ** 2 / Gm == pytest.approx(expect_real, rel=1e-12)
        # attractive: a_0 points towards particle 1, a_1 = -a_0
        assert np.dot(a[0], d) > 0
        assert np.allclose(a[0], -a[1], rtol=1e-13, atol=0)
        assert np.allclose(a[0] / np.linalg.norm(a[0]), d / np.linalg.norm(d), atol=1e-12)


def test_two_particle_cell_distance_cutoff():
    """cells at Chebyshev distance exactly R interact (non-zero force), cells
    at distance R+1 do not interact at all -- exactly zero, however close their corners are."""
    K, R, box, Gm, eps = 8, 2, 1.0, 1.0, 1e-3
    w = box / K
    a_in = oracle.forces(np.array([[0.5 * w, 0.5 * w, 0.5 * w], [2.5 * w, 0.5 * w, 0.5 * w]], np.float32), K, R, eps, box, Gm)
    assert a_in[0, 0] == pytest.approx(Gm / (2 * w) ** 2, rel=1e-12)
    # distance R+1 in cells, but only ~2 cell widths apart in space (far corner to near corner)
    pos = np.array([[0.99 * w, 0.5 * w, 0.5 * w], [3.01 * w, 0.5 * w, 0.5 * w]], np.float32)
    a_out = oracle.forces(pos, K, R, eps, box, Gm)
    assert (a_out == 0).all()
    # periodic: cells 0 and K-2 are at distance 2 through the box edge
    pos = np.array([[0.5 * w, 0.5 * w, 0.5 * w], [0.5 * w, 0.5 * w, (K - 1.5) * w]], np.float32)
    a_per = oracle.forces(pos, K, R, eps, box, Gm)
    assert a_per[0, 2] == pytest.approx(-Gm / (2 * w) ** 2, rel=1e-12)     # pulled across the edge (-z)
    with pytest.raises(ValueError):
        oracle.forces(pos, 4, 2, eps, box, Gm)       # K < 2R+1 would list a cell twice


def test_plummer_two_particle_closed_form():
    """Eq. 1: |a| = Gm r / (r^2 + eps_p^2)^(3/2)."""
    K, R, box, Gm, eps = 6, 2, 3.0, 2.0, 0.05
    for r in (0.01, 0.05, 0.2, 0.45):
        pos = np.array([[1.25, 1.25, 1.25], [1.25 + r, 1.25, 1.25]], np.float32)
        rr = float(pos[1, 0].astype(np.float64) - pos[0, 0].astype(np.float64))
        a = oracle.forces(pos, K, R, eps, box, Gm, softening="plummer")
        assert a[0, 0] == pytest.approx(Gm * rr / (rr * rr + eps * eps) ** 1.5, rel=1e-12)


# ----------------------------------------------------------------------------- brute force
@pytest.mark.parametrize("K,R", [(5, 2), (6, 2), (7, 2), (8, 2), (3, 1), (4, 1), (6, 1)])
def test_against_pair_centric_brute_force(K, R):
    rng = np.random.default_rng(100 * K + R)
    n = 400
    box = 2.5
    pos = (rng.random((n, 3)) * box).astype(np.float32)
    # a clump so that some pairs are inside eps, and a few coincident particles (r = 0)
    pos[:60] = (pos[0] + 0.02 * rng.standard_normal((60, 3))).astype(np.float32) % np.float32(box)
    pos[100] = pos[101]
    pos = np.clip(pos, 0, np.nextafter(np.float32(box), np.float32(0)))
    eps, Gm = 0.03, 1.0 / n
    ref = brute_force(pos, K, R, eps, box, Gm)
    got = oracle.forces(pos, K, R, eps, box, Gm)
    scale = np.sqrt((ref ** 2).sum(axis=1).mean())
    assert np.abs(got - ref).max() < 1e-12 * scale
    # Plummer variant through the same pair set
    refp = brute_force(pos, K, R, eps, box, Gm, softening="plummer")
    gotp = oracle.forces(pos, K, R, eps, box, Gm, softening="plummer")
    assert np.abs(gotp - refp).max() < 1e-12 * scale
    # sink subset, arbitrary order
    idx = rng.permutation(n)[:57]
    sub = oracle.forces(pos, K, R, eps, box, Gm, sink_idx=idx)
    assert np.array_equal(sub, got[idx])


def test_all_pairs_textbook_sum_for_K_equal_2R_plus_1():
    """For K = 2R+1 every cell neighbours every other exactly once, so the near field is the
    all-pairs direct sum with the image fixed by the cell offset; with eps below the smallest
    separation it is the textbook sum of d/|d|^3."""
    rng = np.random.default_rng(7)
    K, R, box, n = 5, 2, 1.0, 300
    pos = rng.random((n, 3)).astype(np.float32)
    x = pos.astype(np.float64)
    c = cells_f32(pos, K, box)
    dc = c[None, :, :] - c[:, None, :]
    img = np.where(dc > R, -1, np.where(dc < -R, 1, 0))
    d = x[None, :, :] + img * box - x[:, None, :]
    r2 = (d ** 2).sum(axis=2)
    np.fill_diagonal(r2, np.inf)
    eps = 0.5 * np.sqrt(r2.min())
    ref = (d / r2[:, :, None] ** 1.5).sum(axis=1) / n
    got = oracle.forces(pos, K, R, eps, box, 1.0 / n)
    assert np.abs(got - ref).max() < 1e-12 * np.abs(ref).max()


# ----------------------------------------------------------------------------- invariants
def _clustered(n, box, rng):
    pos = rng.random((n, 3)) * box
    k = n // 2
    centres = rng.random((8, 3)) * box
    pos[:k] = centres[rng.integers(0, 8, k)] + 0.01 * box * rng.standard_normal((k, 3))
    return np.mod(pos, box).astype(np.float32) % np.float32(box)


def test_zero_net_force_and_antisymmetry():
    """F_ij = -F_ji and the neighbour relation is symmetric => sum_i a_i = 0 (equal masses) on a
    fully periodic box, for any clustering."""
    rng = np.random.default_rng(3)
    pos = _clustered(6000, 1.0, rng)
    pos = np.minimum(pos, np.nextafter(np.float32(1), np.float32(0)))
    a = oracle.forces(pos, 8, 2, 2e-3, 1.0, 1.0 / 6000)
    mag = np.sqrt((a ** 2).sum(axis=1))
    assert np.abs(a.sum(axis=0)).max() < 1e-12 * mag.sum()
    assert mag.max() > 0


def test_symmetric_lattice_gives_zero_force():
    """One particle per cell at the cell centre: the (2R+1)^3 block is point-symmetric about
    every sink, so the near-field force vanishes (the near-field-only special case of the
    homogeneous-lattice test).  For an m^3 sub-lattice per cell the forces are
    mirror-antisymmetric within the cell and sum to zero."""
    K, R, box = 8, 2, 1.0          # power of two: the lattice is exact in float32
    g = (np.arange(K) + 0.5) / K
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float32)
    a = oracle.forces(pos, K, R, 1e-3, box, 1.0)
    assert np.abs(a).max() < 1e-11 * (1.0 / (box / K) ** 2)
    m = 2
    g2 = (np.arange(K * m) + 0.5) / (K * m)
    pos2 = np.stack(np.meshgrid(g2, g2, g2, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float32)
    a2 = oracle.forces(pos2, K, R, 1e-3, box, 1.0).reshape(K * m, K * m, K * m, 3)
    assert np.abs(a2).max() > 1e-3                          # not zero: the near field alone is not
    assert np.abs(a2[0::2, :, :, 0] + a2[1::2, :, :, 0]).max() < 1e-10 * np.abs(a2).max()
    assert np.abs(a2[:, :, 0::2, 2] + a2[:, :, 1::2, 2]).max() < 1e-10 * np.abs(a2).max()


def _quantised(n, rng, bits=18):
    m = rng.integers(0, 1 << bits, size=(n, 3))
    return ((m + 0.5) / float(1 << bits)).astype(np.float32)     # exact in float32, never on a cell face


def test_power_of_two_rescaling_is_bit_exact():
    """Scaling positions, eps and box by 2^k scales every intermediate by a power of two:
    a -> a * 2^(-2k) bit for bit."""
    rng = np.random.default_rng(11)
    pos = _quantised(3000, rng)
    a1 = oracle.forces(pos, 8, 2, 2.0 ** -9, 1.0, 1.0)
    for k in (-3, 5):
        s = 2.0 ** k
        a2 = oracle.forces(pos * np.float32(s), 8, 2, 2.0 ** -9 * s, s, 1.0)
        assert np.array_equal(a2, a1 / s ** 2)


def test_whole_cell_translation_and_mirror_and_permutation():
    rng = np.random.default_rng(12)
    K, R, eps = 8, 2, 2.0 ** -8
    pos = _quantised(3000, rng)
    pos[:500, :] = _quantised(500, rng) / np.float32(16) + np.float32(0.96875 - 1 / 64)  # clump at the box corner
    pos = pos % np.float32(1.0)
    a1 = oracle.forces(pos, K, R, eps, 1.0, 1.0)
    scale = np.sqrt((a1 ** 2).sum(axis=1)).max()
    # (ii) translation by whole cells modulo L exercises every wrap path
    shift = np.array([3, 7, 5], dtype=np.float32) / np.float32(K)
    pos_t = (pos + shift) % np.float32(1.0)
    a_t = oracle.forces(pos_t, K, R, eps, 1.0, 1.0)
    assert np.abs(a_t - a1).max() < 1e-12 * scale
    # (iii) mirror x -> L - x flips a_x
    pos_m = pos.copy(); pos_m[:, 0] = np.float32(1.0) - pos[:, 0]
    a_m = oracle.forces(pos_m, K, R, eps, 1.0, 1.0)
    assert np.abs(a_m[:, 0] + a1[:, 0]).max() < 1e-12 * scale
    assert np.abs(a_m[:, 1:] - a1[:, 1:]).max() < 1e-12 * scale
    # axis permutation x<->z swaps components (catches a transposed axis / wrong key order)
    a_s = oracle.forces(pos[:, ::-1].copy(), K, R, eps, 1.0, 1.0)
    assert np.abs(a_s[:, ::-1] - a1).max() < 1e-12 * scale
    # (iv) permuting the input permutes the output
    p = rng.permutation(pos.shape[0])
    a_p = oracle.forces(pos[p], K, R, eps, 1.0, 1.0)
    assert np.abs(a_p - a1[p]).max() < 1e-12 * scale


# ----------------------------------------------------------------------------- binning
def test_binning_structure_and_stability():
    rng = np.random.default_rng(21)
    K, box, n = 7, 3.0, 5000
    pos = (rng.random((n, 3)) * box).astype(np.float32)
    pos = np.minimum(pos, np.nextafter(np.float32(box), np.float32(0)))
    b = oracle.bin_particles(pos, K, box)
    cnt, off, perm, ps = b["cell_count"], b["cell_offset"], b["perm"], b["pos_sorted"]
    assert b["n_out_of_range"] == 0
    assert cnt.sum() == n and off[0] == 0 and off[-1] == n
    assert np.array_equal(np.diff(off.astype(np.int64)), cnt.astype(np.int64))
    assert np.array_equal(np.sort(perm), np.arange(n))
    c = cells_f32(pos, K, box)
    key = (c[:, 0] * K + c[:, 1]) * K + c[:, 2]                      # x slowest, z fastest
    k2, _ = oracle.keys(pos, K, box)
    assert np.array_equal(k2, key)
    assert np.array_equal(key[perm], np.repeat(np.arange(K ** 3), cnt))   # cell-contiguous, ordered
    # stable: original indices increase within each cell  <=> perm equals a stable argsort
    assert np.array_equal(perm, np.argsort(key, kind="stable"))
    # offsets from own cell centre, |o| <= w/2 (+ rounding)
    w = box / K
    assert np.abs(ps[:, :3]).max() <= 0.5 * w * (1 + 1e-6)
    centre = (c[perm] + 0.5) * w
    assert np.abs(ps[:, :3].astype(np.float64) + centre - pos[perm].astype(np.float64)).max() < 4e-7 * box
    assert (ps[:, 3] == 0).all()


def test_binning_exact_offsets_power_of_two():
    """With power-of-two K and box the cell centres are exact: a particle at (c + 1/4) w has
    offset exactly -w/4 and one at the centre exactly 0."""
    K, box = 16, 1.0
    w = box / K
    c = np.array([[0, 5, 15], [7, 7, 7], [15, 0, 3]])
    pos = np.concatenate([(c + 0.25) * w, (c + 0.5) * w]).astype(np.float32)
    b = oracle.bin_particles(pos, K, box)
    got = np.empty((6, 3), np.float32)
    got[b["perm"]] = b["pos_sorted"][:, :3]
    assert np.array_equal(got[:3], np.full((3, 3), -w / 4, np.float32))
    assert np.array_equal(got[3:], np.zeros((3, 3), np.float32))


def test_binning_edge_cases():
    K, box = 10, 1.0
    top = np.nextafter(np.float32(1.0), np.float32(0))
    pos = np.array([[top, 0.0, 0.5], [1.0, 0.2, 0.2], [-0.1, 0.3, 0.3], [0.0, 0.0, 0.0]], np.float32)
    key, nbad = oracle.keys(pos, K, box)
    assert nbad == 2                                      # x = box and x < 0 are out of range
    assert key[0] == (9 * K + 0) * K + 5                  # x just below box stays in the last cell
    assert key[1] == (9 * K + 2) * K + 2 and key[2] == (0 * K + 3) * K + 3 and key[3] == 0
    b = oracle.bin_particles(np.zeros((0, 3), np.float32), K, box)
    assert b["cell_count"].sum() == 0 and b["cell_offset"][-1] == 0
    # DESIGN.md reading c9: a valid x just below box whose float32 product x * (K / box) rounds up
    # to K (499.99997 * 0.512f == 256.0f) is clamped into cell K-1 and is NOT out of range
    K, box = 256, 500.0
    top = np.nextafter(np.float32(box), np.float32(0))
    assert np.float32(top) * (np.float32(K) / np.float32(box)) == np.float32(K)
    key, nbad = oracle.keys(np.array([[top, top, 1.0], [np.float32(box), 1.0, 1.0]], np.float32), K, box)
    assert nbad == 1 and key[0] == ((K - 1) * K + (K - 1)) * K + 0 and key[1] // (K * K) == K - 1


def test_interaction_count():
    rng = np.random.default_rng(5)
    for K, R in [(5, 2), (7, 2), (6, 1)]:
        pos = rng.random((700, 3)).astype(np.float32)
        b = oracle.bin_particles(pos, K, 1.0)
        c = cells_f32(pos, K, 1.0)
        diff = (c[None, :, :] - c[:, None, :]) % K
        near = ((diff <= R) | (diff >= K - R)).all(axis=2)
        assert oracle.interactions(b["cell_count"], K, R) == int(near.sum())
    cnt = np.full(8 ** 3, 3, np.uint32)
    assert oracle.interactions(cnt, 8, 2) == 8 ** 3 * 9 * 125
    assert oracle.interactions(cnt, 8, 2, 2, 4) == 2 * 64 * 9 * 125


def test_parity_metric():
    ref = np.array([[3.0, 4.0, 0.0], [0.0, 0.0, 0.1]])
    tst = ref + np.array([[0.05, 0, 0], [0, 0.01, 0]])
    rms = np.sqrt((25 + 0.01) / 2)
    e = oracle.parity_error(tst, ref)
    assert e[0] == pytest.approx(0.05 / 5.0) and e[1] == pytest.approx(0.01 / rms)


# ------------------------------------------------- next rows: masses, a_max
def test_masses_two_particle_and_momentum():
    """Unequal masses: the pair force is G m_i m_j F (PAPER.md:37 with Eq. 2), so a_i carries m_j.
    Two particles: |a_0| / |a_1| = m_1 / m_0 and each is m_other times the closed form; many
    particles: total momentum change sum_i m_i a_i = 0 on a fully periodic box."""
    eps, box, K = 0.01, 1.0, 8
    d = np.array([0.3, -0.4, 0.5]) / np.sqrt(0.5) * 0.5 * eps        # |d| = eps/2: u s(u) = 2 (golden value)
    pos = np.array([[0.51, 0.52, 0.53], [0.51, 0.52, 0.53] + d], dtype=np.float32)
    m = np.array([3.0, 0.25], dtype=np.float32)
    a = oracle.forces(pos, K, 2, eps, box, 1.0, mass=m)
    sep = pos[1].astype(np.float64) - pos[0].astype(np.float64)
    r = np.sqrt((sep ** 2).sum())
    u = r / eps
    closed = (10 - 15 * u + 6 * u * u) * r / eps ** 3
    assert np.allclose(a[0], 0.25 * closed * sep / r, rtol=1e-12)
    assert np.allclose(a[1], -3.0 * closed * sep / r, rtol=1e-12)
    rng = np.random.default_rng(11)
    pos = _clustered(4000, 1.0, rng)
    pos = np.minimum(pos, np.nextafter(np.float32(1), np.float32(0)))
    m = rng.uniform(0.1, 5.0, 4000).astype(np.float32)
    a = oracle.forces(pos, 8, 2, 2e-3, 1.0, 1.0, mass=m)
    p = (m.astype(np.float64)[:, None] * a)
    assert np.abs(p.sum(axis=0)).max() < 1e-11 * np.sqrt((p ** 2).sum(axis=1)).sum()


def test_masses_against_brute_force_and_superposition():
    """Brute force with masses (no cell lists), equal masses == the scalar-Gm path, and linearity
    in the source masses: a[m1 + m2] = a[m1] + a[m2]."""
    rng = np.random.default_rng(12)
    n, K, R, eps, box = 300, 6, 2, 0.05, 1.0
    pos = rng.random((n, 3)).astype(np.float32)
    m1 = rng.uniform(0.0, 2.0, n).astype(np.float32)
    m2 = rng.uniform(0.0, 2.0, n).astype(np.float32)
    x = pos.astype(np.float64)
    c = cells_f32(pos, K, box)
    ref = np.zeros((n, 3))
    for i in range(n):
        for j in range(n):
            dl = []
            for ax in range(3):
                df = (c[j, ax] - c[i, ax]) % K
                dl.append(df if df <= R else (df - K if df >= K - R else None))
            if None in dl:
                continue
            img = [(c[i, ax] + dl[ax] - c[j, ax]) // K for ax in range(3)]
            dv = x[j] + np.array(img) * box - x[i]
            r = np.sqrt((dv ** 2).sum())
            if r == 0:
                continue
            u = r / eps
            f = (10 - 15 * u + 6 * u * u) / eps ** 3 if u < 1 else 1 / r ** 3
            ref[i] += float(m1[j]) * f * dv
    a1 = oracle.forces(pos, K, R, eps, box, 1.0, mass=m1)
    assert np.allclose(a1, ref, rtol=1e-10, atol=1e-10 * np.abs(ref).max())
    a2 = oracle.forces(pos, K, R, eps, box, 1.0, mass=m2)
    a12 = oracle.forces(pos, K, R, eps, box, 1.0, mass=(m1.astype(np.float64) + m2).astype(np.float32))
    # m1 + m2 is rounded to float32 once: compare with the same rounded masses split exactly
    m12 = (m1.astype(np.float64) + m2).astype(np.float32)
    a2x = oracle.forces(pos, K, R, eps, box, 1.0, mass=(m12.astype(np.float64) - m1).astype(np.float32))
    assert np.allclose(a12, a1 + a2x, rtol=1e-6, atol=1e-6 * np.abs(a12).max())
    assert np.abs(a2).max() > 0
    eq = oracle.forces(pos, K, R, eps, box, 1.0, mass=np.full(n, 0.5, np.float32))
    assert np.allclose(eq, oracle.forces(pos, K, R, eps, box, 0.5), rtol=1e-13, atol=0)


def test_cell_amax_definition():
    """Per-cell max |a| against a python loop; empty cells are 0; the maximum
    over cells is the global maximum."""
    rng = np.random.default_rng(13)
    n, K = 500, 5
    pos = rng.random((n, 3)).astype(np.float32)
    a = oracle.forces(pos, K, 2, 0.02, 1.0, 1.0 / n)
    key, _ = oracle.keys(pos, K, 1.0)
    got = oracle.cell_amax(a, key, K ** 3)
    mag = np.sqrt((a ** 2).sum(axis=1))
    ref = np.zeros(K ** 3)
    for i in range(n):
        ref[key[i]] = max(ref[key[i]], mag[i])
    assert np.array_equal(got, ref)
    assert got.max() == mag.max()
    assert (got[np.bincount(key, minlength=K ** 3) == 0] == 0).all()


# ------------------------------------------------- next rows: kick, drift
def test_kick_drift_closed_forms_and_wrap():
    """Exactly representable cases worked by hand (box = 1): the velocity is updated FIRST and the
    drift uses the new velocity; one periodic wrap either way; x + box rounding up to box gives 0."""
    pos = np.array([[0.25, 0.875, 0.125]], np.float32)
    vel = np.array([[0.5, 1.0, -1.0]], np.float32)
    acc = np.array([[1.0, 0.0, 0.0]], np.float32)
    x, v = oracle.kick_drift(pos, vel, acc, 0.5, 0.25, 1.0)
    # x: v1 = 0.5 + 1*0.5 = 1.0, x1 = 0.25 + 1.0*0.25 = 0.5 (an update with the OLD v would give 0.375)
    # y: 0.875 + 0.25 = 1.125 -> 0.125;  z: 0.125 - 0.25 = -0.125 -> 0.875
    assert np.array_equal(v, np.array([[1.0, 1.0, -1.0]], np.float32))
    assert np.array_equal(x, np.array([[0.5, 0.125, 0.875]], np.float32))
    tiny = np.array([[-1e-12, 0.0, 0.0]], np.float32)
    x, _ = oracle.kick_drift(tiny, np.zeros((1, 3), np.float32), np.zeros((1, 3), np.float32), 0.0, 0.0, 1.0)
    assert x[0, 0] == 0.0                      # -1e-12 + 1 rounds to 1.0f == box -> 0
    assert (x >= 0).all() and (x < 1).all()


def test_kick_drift_is_symplectic_leapfrog():
    """Harmonic oscillator a = -x stepped with (kick h, drift h): the leapfrog map conserves the
    modified energy v^2 + x^2 - h x v exactly in real arithmetic (textbook), so over 10^4 steps it
    stays within float32 rounding drift, while x^2 + v^2 oscillates by O(h).  A drift with the old
    velocity (explicit Euler) would grow by (1 + h^2) per step."""
    h, box = 0.05, 8.0
    x = np.array([[4.0 + 1.0, 4.0, 4.0]], np.float32)      # oscillate about the box centre
    v = np.zeros((1, 3), np.float32)
    inv0 = None
    for _ in range(10000):
        a = -(x - np.float32(4.0))
        x, v = oracle.kick_drift(x, v, a, h, h, box)
        q = float(x[0, 0]) - 4.0
        inv = float(v[0, 0]) ** 2 + q * q - h * q * float(v[0, 0])
        inv0 = inv if inv0 is None else inv0
        assert abs(inv - inv0) < 2e-3 * inv0
    assert abs(inv0 - 1.0) < 0.01


def test_cell_vrms_definition():
    rng = np.random.default_rng(21)
    n, K = 700, 4
    pos = rng.random((n, 3)).astype(np.float32)
    vel = rng.standard_normal((n, 3)).astype(np.float32)
    key, _ = oracle.keys(pos, K, 1.0)
    got, vmax = oracle.cell_vrms(vel, key, K ** 3)
    v64 = vel.astype(np.float64)
    for c in range(K ** 3):
        sel = key == c
        ref = np.sqrt((v64[sel] ** 2).sum(axis=1).mean()) if sel.any() else 0.0
        assert abs(got[c] - ref) <= 1e-14 * max(ref, 1.0)
    assert vmax == np.abs(v64).max()
    # equal speeds in every direction: v_rms is that speed
    u = rng.standard_normal((n, 3))
    u = (3.0 * u / np.sqrt((u ** 2).sum(axis=1))[:, None]).astype(np.float32)
    got, _ = oracle.cell_vrms(u, key, K ** 3)
    assert np.allclose(got[np.bincount(key, minlength=K ** 3) > 0], 3.0, rtol=1e-6)


def test_timestep_terms_hand_worked():
    """Criteria 2 and 3 on a box worked by hand.  Four cells: A (n = 2, v_rms = 3,
    a_max = 6), B (n = 6, v_rms = 1, a_max = 0.5), C empty, D (n = 2, v_rms = 2, a_max = 0: no ratio).
    Cell ratios 0.5 and 2; global v_rms = sqrt((2*9 + 6*1 + 2*4) / 10) = sqrt(3.2); global a_max = 6."""
    t = oracle.timestep_terms([3, 1, 7, 2], [6, 0.5, 9, 0], [2, 6, 0, 2], K=4, box=2.0, vmax=0.25)
    assert t["cells_used"] == 2
    assert t["ratio_cell_min"] == 0.5 and t["ratio_cell_max"] == 2.0
    assert abs(t["vrms_global"] - np.sqrt(3.2)) < 1e-15
    assert t["amax_global"] == 6.0                    # the empty cell's stale entries (7, 9) take no part
    assert abs(t["ratio_global"] - np.sqrt(3.2) / 6.0) < 1e-15
    # "use the maximum of the global and cell-based values ... protects us from ... abnormally cold cells": a cold
    # cell (small v_rms, large a_max) must not shorten the step below the global value
    assert t["ratio_criterion2"] == t["ratio_cell_min"] == 0.5        # here the cell value (0.5) exceeds the global 0.298
    cold = oracle.timestep_terms([3, 1e-6, 7, 2], [6, 0.5, 9, 0], [2, 6, 0, 2], K=4, box=2.0, vmax=0.25)
    assert cold["ratio_cell_min"] < 1e-5 and cold["ratio_criterion2"] == cold["ratio_global"]
    # criterion 3: 0.8 * cell width / vmax = 0.8 * 0.5 / 0.25
    assert abs(t["drift_limit"] - 1.6) < 1e-15
    assert oracle.timestep_terms([1], [1], [1], K=1, box=1.0)["drift_limit"] == float("inf")
