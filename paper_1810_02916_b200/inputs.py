"""Seeded synthetic inputs for the five BASELINE.json configs (C1..C5).

This module holds NO arithmetic of the method (no cell assignment, no force law); it only
draws positions.  Both the CUDA path and the CPU oracle receive the SAME arrays produced
here -- the arrays, not the generator, are the contract.  The
paper's own workload is the S2016 Euclid comparison box, which is not
available offline; C4 and C5 take its shape (500 h^-1 Mpc periodic box, eps = 10 h^-1 kpc,
strongly uneven cells) and stand in for it.

Generation is chunked (fixed chunk of 2^22 particles, one torch.Generator per chunk seeded
from (seed, chunk index)) so that 2^30 particles can be produced on the GPU without a
second full-size buffer, and so that a prefix of a config equals the same prefix of a
larger run.  Halo membership is drawn per particle (multinomial), so input order carries
no structure and no shuffle pass is needed.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Callable, List, Optional

import torch

BASE_SEED = 181002916
CHUNK = 1 << 22


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    N: int              # particles (C5: mean particles per plane x planes, informational)
    K: int              # cells per side
    R: int              # near-field radius in cells
    box: float          # periodic box length L
    eps: float          # spline softening eps_s of Eq. 2 (reading c4)
    Gm: float           # G * m, equal masses
    seed: int
    kind: str           # uniform | lattice | clustered | slab
    # clustered / slab parameters
    frac_halo: float = 0.0
    n_halos: int = 0
    a_lo: float = 0.0   # Plummer scale radius range (log-uniform)
    a_hi: float = 0.0
    r_trunc: float = 0.0
    lattice_n: int = 0
    lattice_sigma: float = 0.0
    # slab (C5)
    planes: int = 0     # sink planes P
    plane0: int = 0     # x index of the first ghost plane
    density_n: int = 0  # particles per box side of the parent box (2048)


def config(which: int) -> Config:
    """The five configs of BASELINE.json, with the open choices of SURVEY.md Sec. 8(d)."""
    s = BASE_SEED + which
    if which == 1:
        N = 32 ** 3
        return Config("C1-uniform-32^3", N, 8, 2, 1.0, 0.025 / 32, 1.0 / N, s, "uniform")
    if which == 2:
        N = 128 ** 3
        return Config("C2-lattice-128^3", N, 32, 2, 1.0, (1.0 / 40) / 128, 1.0 / N, s, "lattice",
                      lattice_n=128, lattice_sigma=0.2 / 128)
    if which == 3:
        N = 256 ** 3
        return Config("C3-clustered-256^3", N, 64, 2, 1.0, (1.0 / 40) / 256, 1.0 / N, s, "clustered",
                      frac_halo=0.5, n_halos=4096, a_lo=0.15 / 64, a_hi=0.15 / 64, r_trunc=2.0 / 64)
    if which == 4:
        N = 1024 ** 3
        return Config("C4-clustered-1024^3", N, 256, 2, 500.0, 0.01, 1.0 / N, s, "clustered",
                      frac_halo=0.4, n_halos=1 << 20, a_lo=0.020, a_hi=0.300,
                      r_trunc=2.0 * 500.0 / 256)
    if which == 5:
        N = 2048 ** 3
        return Config("C5-slab-2048^3-density", N, 512, 2, 500.0, 0.01, 1.0 / N, s, "slab",
                      frac_halo=0.4, n_halos=1 << 20, a_lo=0.020, a_hi=0.300,
                      r_trunc=2.0 * 500.0 / 256, planes=16, plane0=100, density_n=2048)
    if which == 6:
        # not a BASELINE.json config: the dense-cell end of the range ("the largest cell has
        # over 200,000 particles"): one cell of ~4x10^5 particles in an otherwise almost empty K = 5 box
        N = 400_000
        return Config("D1-one-dense-cell-4e5", N, 5, 2, 1.0, 0.01 * 0.2, 1.0 / N, s, "onecell")
    if which == 7:
        # not a BASELINE.json config: the C3 recipe on a grid four times coarser -- 4096 particles per cell on average, 254
        # cells of >= 4096 (the largest 1.2x10^5) holding half the particles and neighbouring one another: the tree near
        # field (nf_forces_tree) with many trees
        return scaled(dataclasses.replace(config(3), seed=s), 256 ** 3, 16, name="D2-clustered-256^3-K16")
    raise ValueError("config number must be 1..5 (6: the one-dense-cell profiling workload, 7: many dense cells)")


def scaled(cfg: Config, N: int, K: int, name: Optional[str] = None) -> Config:
    """Same recipe at another size, keeping ~N/K^3 particles per cell and eps relative to the
    mean interparticle spacing; halo count scales with the number of cells.  Used by the
    parity tests for sizes the oracle finishes in seconds."""
    spacing_old = cfg.box / round(cfg.N ** (1 / 3))
    spacing_new = cfg.box / (N ** (1 / 3))
    w_old, w_new = cfg.box / cfg.K, cfg.box / K
    kw = dict(N=N, K=K, eps=cfg.eps * spacing_new / spacing_old, Gm=1.0 / N,
              name=name or f"{cfg.name}@N={N},K={K}")
    if cfg.kind in ("clustered", "slab"):
        kw.update(n_halos=max(1, int(round(cfg.n_halos * (K / cfg.K) ** 3))),
                  a_lo=cfg.a_lo * w_new / w_old, a_hi=cfg.a_hi * w_new / w_old,
                  r_trunc=cfg.r_trunc * w_new / w_old)
    if cfg.kind == "lattice":
        n = round(N ** (1 / 3))
        kw.update(lattice_n=n, lattice_sigma=0.2 * cfg.box / n)
    return dataclasses.replace(cfg, **kw)


def _gen(seed: int, chunk: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed((seed * 1000003 + chunk * 7919 + 12345) & 0x7FFFFFFFFFFFFFFF)
    return g


def _wrap_(x: torch.Tensor, box: float) -> torch.Tensor:
    """Periodic wrap into [0, box) in float32, guarding the x == box rounding case."""
    x -= torch.floor(x / box) * box
    x[x >= box] = 0.0
    x[x < 0] = 0.0
    return x


def _plummer_offsets(n: int, a: torch.Tensor, r_trunc: float, g: torch.Generator, device) -> torch.Tensor:
    """n isotropic displacement vectors from a Plummer sphere of scale radius a (tensor [n]),
    truncated at r_trunc: r = a / sqrt(X^(-2/3) - 1), X uniform on (0, X_t),
    X_t = M(<r_t)/M = r_t^3 / (r_t^2 + a^2)^(3/2)."""
    a64 = a.double()
    xt = (r_trunc ** 3) / (r_trunc ** 2 + a64 ** 2) ** 1.5
    u = torch.rand(n, generator=g, device=device, dtype=torch.float64)
    X = (u * (1.0 - 1e-12) + 1e-12) * xt
    r = a64 / torch.sqrt(X ** (-2.0 / 3.0) - 1.0)
    cost = torch.rand(n, generator=g, device=device, dtype=torch.float64) * 2.0 - 1.0
    phi = torch.rand(n, generator=g, device=device, dtype=torch.float64) * (2.0 * math.pi)
    sint = torch.sqrt(torch.clamp(1.0 - cost * cost, min=0.0))
    return torch.stack([r * sint * torch.cos(phi), r * sint * torch.sin(phi), r * cost], dim=1)


def _halo_catalogue(cfg: Config, device):
    """Halo centres (uniform in the box) and scale radii (log-uniform in [a_lo, a_hi])."""
    g = _gen(cfg.seed, -1, device)
    centres = torch.rand(cfg.n_halos, 3, generator=g, device=device, dtype=torch.float64) * cfg.box
    if cfg.a_hi > cfg.a_lo:
        la = torch.rand(cfg.n_halos, generator=g, device=device, dtype=torch.float64)
        scales = cfg.a_lo * (cfg.a_hi / cfg.a_lo) ** la
    else:
        scales = torch.full((cfg.n_halos,), cfg.a_lo, device=device, dtype=torch.float64)
    return centres, scales


def make_positions(cfg: Config, device="cpu", out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """float32 [N, 3] positions in [0, box)^3 for configs of kind uniform / lattice / clustered."""
    device = torch.device(device)
    N = cfg.N
    if out is None:
        out = torch.empty(N, 3, dtype=torch.float32, device=device)
    assert out.shape == (N, 3) and out.dtype == torch.float32
    cat = _halo_catalogue(cfg, device) if cfg.kind == "clustered" else None
    for c, lo in enumerate(range(0, N, CHUNK)):
        out[lo:min(N, lo + CHUNK)] = make_positions_chunk(cfg, c, device, cat)
    return out


def make_positions_chunk(cfg: Config, c: int, device="cpu", catalogue=None) -> torch.Tensor:
    """Chunk c (particles [c*CHUNK, min(N, (c+1)*CHUNK))) of make_positions: every chunk has its own
    generator, so a rank of a sharded run can produce any part of the box without the rest."""
    device = torch.device(device)
    lo = c * CHUNK
    assert 0 <= lo < cfg.N
    hi = min(cfg.N, lo + CHUNK)
    n = hi - lo
    g = _gen(cfg.seed, c, device)
    if cfg.kind == "uniform":
        x = torch.rand(n, 3, generator=g, device=device, dtype=torch.float32) * cfg.box
    elif cfg.kind == "lattice":
        m = cfg.lattice_n
        idx = torch.arange(lo, hi, device=device, dtype=torch.int64)
        ijk = torch.stack([idx // (m * m), (idx // m) % m, idx % m], dim=1).double()
        x = (ijk + 0.5) * (cfg.box / m)
        x = x + torch.randn(n, 3, generator=g, device=device, dtype=torch.float64) * cfg.lattice_sigma
        x = x.float()
    elif cfg.kind == "clustered":
        centres, scales = catalogue if catalogue is not None else _halo_catalogue(cfg, device)
        x = torch.rand(n, 3, generator=g, device=device, dtype=torch.float64) * cfg.box
        is_halo = torch.rand(n, generator=g, device=device, dtype=torch.float64) < cfg.frac_halo
        hid = torch.randint(0, cfg.n_halos, (n,), generator=g, device=device)
        off = _plummer_offsets(n, scales[hid], cfg.r_trunc, g, device)
        x = torch.where(is_halo[:, None], centres[hid] + off, x).float()
    elif cfg.kind == "onecell":
        # Normal(centre of the middle cell, 0.08 w) clipped into that cell; the first 1000 particles uniform in the box
        w = cfg.box / cfg.K
        mid = (cfg.K // 2 + 0.5) * w
        x = mid + 0.08 * w * torch.randn(n, 3, generator=g, device=device, dtype=torch.float64)
        x = x.clamp(mid - 0.49 * w, mid + 0.49 * w)
        u = torch.rand(n, 3, generator=g, device=device, dtype=torch.float64) * cfg.box
        first = (torch.arange(lo, hi, device=device) < 1000)[:, None]
        x = torch.where(first, u, x).float()
    else:
        raise ValueError(f"make_positions: kind {cfg.kind!r} not supported (use make_slab_planes)")
    return _wrap_(x, cfg.box)


def make_slab_planes(cfg: Config, device="cpu", n_planes_total: Optional[int] = None,
                     density_scale: float = 1.0, plane_of: Optional[Callable[[torch.Tensor], torch.Tensor]] = None
                     ) -> List[torch.Tensor]:
    """C5: the particles of P + 2R consecutive x-planes (plane0 .. plane0+P+2R-1; the outer R on
    each side are ghosts) of a density_n^3-particle periodic box with the C4-style halo
    catalogue.  Returns one float32 [n_p, 3] tensor per plane (global coordinates, arbitrary
    in-plane order).  density_scale < 1 thins the box for small tests.

    ``plane_of(x)`` maps float32 [n, 3] positions to the int64 x-plane (x-cell index) each particle
    is filed under.  Which plane a particle on or next to a plane face belongs to is decided by the
    float32 cell-assignment formula of the method, which this module must not restate: the caller
    passes the method's own answer (tests: the oracle's keys // K^2; bench.py: the library's nf_keys
    // K^2).  Particles filed outside the chunk's planes are left out; nothing else is dropped."""
    assert cfg.kind == "slab"
    assert plane_of is not None, "make_slab_planes needs plane_of (the method's cell assignment); see the docstring"
    device = torch.device(device)
    P2 = n_planes_total if n_planes_total is not None else cfg.planes + 2 * cfg.R
    w = cfg.box / cfg.K
    x0, x1 = cfg.plane0 * w, (cfg.plane0 + P2) * w
    assert cfg.plane0 >= 0 and cfg.plane0 + P2 <= cfg.K, "chunk must not wrap in x"
    n_box = float(cfg.density_n) ** 3 * density_scale
    g = _gen(cfg.seed, -2, device)
    parts = []
    # uniform component: Poisson number in the chunk volume
    lam = (1.0 - cfg.frac_halo) * n_box * (x1 - x0) / cfg.box
    n_uni = int(torch.poisson(torch.tensor([lam], dtype=torch.float64), generator=_gen(cfg.seed, -3, "cpu")).item())
    for c, lo in enumerate(range(0, n_uni, CHUNK)):
        n = min(CHUNK, n_uni - lo)
        gg = _gen(cfg.seed, 1000 + c, device)
        x = torch.rand(n, 3, generator=gg, device=device, dtype=torch.float64)
        x[:, 0] = x0 + x[:, 0] * (x1 - x0)
        x[:, 1:] *= cfg.box
        parts.append(x.float())
    # halo component: halos whose truncated sphere can reach the chunk
    centres, scales = _halo_catalogue(cfg, device)
    near = (centres[:, 0] > x0 - cfg.r_trunc) & (centres[:, 0] < x1 + cfg.r_trunc)
    hsel = torch.nonzero(near).flatten()
    per_halo = cfg.frac_halo * n_box / cfg.n_halos
    counts = torch.poisson(torch.full((hsel.numel(),), per_halo, dtype=torch.float64, device=device), generator=g).long()
    hid_all = torch.repeat_interleave(hsel, counts)
    for c, lo in enumerate(range(0, hid_all.numel(), CHUNK)):
        hid = hid_all[lo:lo + CHUNK]
        gg = _gen(cfg.seed, 2000 + c, device)
        off = _plummer_offsets(hid.numel(), scales[hid], cfg.r_trunc, gg, device)
        xh = (centres[hid] + off).float()
        # a coarse geometric pre-cut one cell wider than the chunk (halo members far outside it are of no
        # use); the filing below decides which plane, if any, every survivor belongs to
        xh = xh[(xh[:, 0] >= x0 - w) & (xh[:, 0] < x1 + w)]
        parts.append(xh)
    x = torch.cat(parts, dim=0) if parts else torch.empty(0, 3, dtype=torch.float32, device=device)
    x[:, 1:] = _wrap_(x[:, 1:].contiguous(), cfg.box)
    x = x[(x[:, 0] >= 0) & (x[:, 0] < cfg.box)]
    p = plane_of(x).to(device=device, dtype=torch.int64) - cfg.plane0
    keep = (p >= 0) & (p < P2)
    x, p = x[keep], p[keep]
    # shuffle so in-plane order carries no structure, then split
    perm = torch.randperm(x.shape[0], generator=g, device=device)
    x, p = x[perm], p[perm]
    order = torch.argsort(p, stable=True)
    x, p = x[order], p[order]
    cnt = torch.bincount(p, minlength=P2).tolist()
    planes, s = [], 0
    for n in cnt:
        planes.append(x[s:s + n].contiguous())
        s += n
    return planes


def select_box(pos: torch.Tensor, lo, hi, box: float) -> torch.Tensor:
    """Indices of the particles whose coordinates lie in the periodic axis-aligned box
    [lo, hi) (per axis, lo may be negative and hi may exceed `box`; hi - lo < box).  A plain
    geometric filter used to cut samples out of the big configs for the CPU oracle; it does no
    cell assignment."""
    mask = torch.ones(pos.shape[0], dtype=torch.bool, device=pos.device)
    for ax in range(3):
        x = pos[:, ax]
        l, h = float(lo[ax]), float(hi[ax])
        assert h - l < box
        l_w, h_w = l % box, h % box
        if l_w < h_w:
            mask &= (x >= l_w) & (x < h_w)
        else:
            mask &= (x >= l_w) | (x < h_w)
    return torch.nonzero(mask).flatten()


def clumps(seed: int, K: int, box: float, clumps_, n_bg: int):
    """Seeded numpy test input for dense cells: uniform balls inside chosen cells plus a uniform background.
    clumps_: list of (cell (cx, cy, cz), n, radius in cell widths, centre offset in cell widths).  float32 [N, 3],
    shuffled.  (The late-time state of PAPER.md:75 in miniature: a few cells with thousands of particles.)"""
    import numpy as np
    rng = np.random.default_rng(seed)
    w = box / K
    parts = [rng.random((n_bg, 3)) * box]
    for (c, n, rad, ctr) in clumps_:
        d = rng.normal(size=(n, 3))
        d *= (rng.random(n) ** (1.0 / 3.0) / np.linalg.norm(d, axis=1))[:, None] * rad * w
        parts.append((np.array(c) + 0.5 + np.array(ctr)) * w + d)
    pos = np.concatenate(parts) % box
    return np.ascontiguousarray(pos[rng.permutation(pos.shape[0])], dtype=np.float32)
