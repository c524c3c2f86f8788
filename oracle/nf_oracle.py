"""ctypes loader for oracle/nf_oracle.c -- the plain double-precision CPU oracle.

TEST INFRASTRUCTURE, NOT THE PRODUCT (see the header of nf_oracle.c).  Every function here
is a thin marshalling layer over the C functions of the same name (prefix ``nfo_``); the
arithmetic lives in nf_oracle.c, each routine citing the PAPER.md passage it follows.

Parity status: every function is pinned by tests/test_oracle_pins.py (brute force, closed
forms, invariants); nothing here is "parity unpinned" except kick_drift against the paper (it prints no
formula; pinned to the textbook leapfrog, reading c20).  timestep_terms (criteria 2 and 3,
PAPER.md:193-195, :207) is plain numpy in this file and pinned by a hand-worked four-cell box; which
extremum over cells criterion 2 takes is DESIGN.md reading c19.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nf_oracle.c")
_LIB = os.path.join(_HERE, "libnf_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile nf_oracle.c with gcc (-ffp-contract=off: the float32 binning formulas are a
    bit-exact contract and must not be fused)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        c_f32p = ctypes.POINTER(ctypes.c_float)
        c_u32p = ctypes.POINTER(ctypes.c_uint32)
        c_u64p = ctypes.POINTER(ctypes.c_uint64)
        c_i64p = ctypes.POINTER(ctypes.c_int64)
        c_f64p = ctypes.POINTER(ctypes.c_double)
        lib.nfo_keys.restype = ctypes.c_int64
        lib.nfo_keys.argtypes = [c_f32p, ctypes.c_int64, ctypes.c_int, ctypes.c_float, c_u32p]
        lib.nfo_bin.restype = ctypes.c_int64
        lib.nfo_bin.argtypes = [c_f32p, ctypes.c_int64, ctypes.c_int, ctypes.c_float,
                                c_f32p, c_u32p, c_u32p, c_u64p]
        lib.nfo_forces.restype = ctypes.c_int
        lib.nfo_forces.argtypes = [c_f32p, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                   ctypes.c_float, ctypes.c_double, c_i64p, ctypes.c_int64,
                                   ctypes.c_int, ctypes.c_int, c_f64p]
        lib.nfo_forces_m.restype = ctypes.c_int
        lib.nfo_forces_m.argtypes = [c_f32p, c_f32p, ctypes.c_int64, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                     ctypes.c_float, ctypes.c_double, c_i64p, ctypes.c_int64,
                                     ctypes.c_int, ctypes.c_int, c_f64p]
        lib.nfo_cell_amax.restype = None
        lib.nfo_cell_amax.argtypes = [c_f64p, c_u32p, ctypes.c_int64, ctypes.c_int64, c_f64p]
        lib.nfo_kick_drift.restype = None
        lib.nfo_kick_drift.argtypes = [c_f32p, c_f32p, c_f32p, ctypes.c_int64, ctypes.c_float, ctypes.c_float, ctypes.c_float]
        lib.nfo_cell_vrms.restype = None
        lib.nfo_cell_vrms.argtypes = [c_f32p, c_u32p, ctypes.c_int64, ctypes.c_int64, c_f64p, c_f64p]
        lib.nfo_interactions.restype = ctypes.c_int64
        lib.nfo_interactions.argtypes = [c_u32p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.nfo_spline_over_r.restype = ctypes.c_double
        lib.nfo_spline_over_r.argtypes = [ctypes.c_double, ctypes.c_double]
        lib.nfo_plummer_over_r.restype = ctypes.c_double
        lib.nfo_plummer_over_r.argtypes = [ctypes.c_double, ctypes.c_double]
        lib.nfo_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _f32(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(ctypes.POINTER(ctypes.c_float))


def max_threads() -> int:
    return int(_load().nfo_max_threads())


def keys(pos, K: int, box: float):
    """Cell key per particle; returns (keys uint32[N], n_out_of_range)."""
    lib = _load()
    pos, p = _f32(pos)
    n = pos.shape[0]
    out = np.empty(n, dtype=np.uint32)
    nbad = lib.nfo_keys(p, n, int(K), float(box), out.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)))
    return out, int(nbad)


def bin_particles(pos, K: int, box: float):
    """Stable counting sort by cell.
    Returns dict(pos_sorted float32[N,4], perm uint32[N], cell_count uint32[K^3],
    cell_offset uint64[K^3+1], n_out_of_range)."""
    lib = _load()
    pos, p = _f32(pos)
    n = pos.shape[0]
    ncell = int(K) ** 3
    ps = np.empty((n, 4), dtype=np.float32)
    perm = np.empty(n, dtype=np.uint32)
    cnt = np.empty(ncell, dtype=np.uint32)
    off = np.empty(ncell + 1, dtype=np.uint64)
    nbad = lib.nfo_bin(p, n, int(K), float(box),
                       ps.ctypes.data_as(ctypes.POINTER(ctypes.c_float)),
                       perm.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)),
                       cnt.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)),
                       off.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)))
    return dict(pos_sorted=ps, perm=perm, cell_count=cnt, cell_offset=off, n_out_of_range=int(nbad))


def forces(pos, K: int, R: int, eps: float, box: float, Gm: float, sink_idx=None,
           softening: str = "spline", nthreads: int = 0, mass=None):
    """Near-field accelerations in double (Eq. 2 :243 / Eq. 1 :233).
    Returns float64[n_sinks, 3] in the order of sink_idx (all particles, input order, if None).
    mass: None = equal masses (Gm = G*m); else float32[N] source masses and Gm = G."""
    lib = _load()
    pos, p = _f32(pos)
    n = pos.shape[0]
    if sink_idx is None:
        sp, ns = None, n
    else:
        sink_idx = np.ascontiguousarray(sink_idx, dtype=np.int64)
        sp, ns = sink_idx.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), sink_idx.shape[0]
    acc = np.zeros((ns, 3), dtype=np.float64)
    soft = {"spline": 0, "plummer": 1}[softening]
    mp = None
    if mass is not None:
        mass = np.ascontiguousarray(mass, dtype=np.float32)
        assert mass.shape == (n,)
        mp = mass.ctypes.data_as(ctypes.POINTER(ctypes.c_float))
    rc = lib.nfo_forces_m(p, mp, n, int(K), int(R), float(eps), float(box), float(Gm), sp, ns, soft,
                          int(nthreads), acc.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    if rc != 0:
        raise ValueError("nfo_forces: bad arguments (need K >= 2R+1, R >= 0, eps > 0, box > 0)")
    return acc


def cell_amax(acc, key, ncell: int):
    """Per-cell maximum of |a|; acc float64[N,3] in input order, key uint32[N]."""
    lib = _load()
    acc = np.ascontiguousarray(acc, dtype=np.float64)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(int(ncell), dtype=np.float64)
    lib.nfo_cell_amax(acc.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), key.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)),
                      acc.shape[0], int(ncell), out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    return out


def kick_drift(pos, vel, acc, kick: float, drift: float, box: float):
    """v <- v + a*kick; x <- wrap(x + v*drift) with the new v (Table 1 "Kick", "Drift"),
    in the float32 contract of DESIGN.md.  Returns new (pos, vel) float32 arrays; inputs are not modified."""
    lib = _load()
    pos = np.array(pos, dtype=np.float32, order="C", copy=True)
    vel = np.array(vel, dtype=np.float32, order="C", copy=True)
    acc = np.ascontiguousarray(acc, dtype=np.float32)
    assert pos.shape == vel.shape == acc.shape and pos.ndim == 2 and pos.shape[1] == 3
    f = ctypes.POINTER(ctypes.c_float)
    lib.nfo_kick_drift(pos.ctypes.data_as(f), vel.ctypes.data_as(f), acc.ctypes.data_as(f), pos.shape[0],
                       float(kick), float(drift), float(box))
    return pos, vel


def cell_vrms(vel, key, ncell: int):
    """(per-cell rms speed float64[ncell], max |v_axis|) -- PAPER.md:193-195."""
    lib = _load()
    vel = np.ascontiguousarray(vel, dtype=np.float32)
    key = np.ascontiguousarray(key, dtype=np.uint32)
    out = np.zeros(int(ncell), dtype=np.float64)
    vmax = ctypes.c_double(0.0)
    lib.nfo_cell_vrms(vel.ctypes.data_as(ctypes.POINTER(ctypes.c_float)), key.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)),
                      vel.shape[0], int(ncell), out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), ctypes.byref(vmax))
    return out, float(vmax.value)


def timestep_terms(cell_vrms, cell_amax, cell_count, K: int, box: float, vmax=None) -> dict:
    """Time-step criteria 2 and 3 written out, plain numpy.  Criterion 2: the step is
    TimeStepAccel times a ratio v_rms / a_max; "we also compute a global v_rms/a_max and use the maximum of the global
    and cell-based values.  This protects us from taking catastrophically small time steps as a result of abnormally
    cold cells" -- a cold cell has a SMALL ratio, so the cell-based value is the minimum over cells (DESIGN.md reading
    c19; the maximum over cells, the literal reading of :194, is returned beside it).  Each cell ratio is the float32
    quotient; cells that are empty or have a_max = 0 are left out.  Criterion 3: step * vmax < 0.8 cell widths."""
    v = np.asarray(cell_vrms, dtype=np.float32).ravel()
    a = np.asarray(cell_amax, dtype=np.float32).ravel()
    n = np.asarray(cell_count, dtype=np.int64).ravel()
    use = (n > 0) & (a > 0)
    q = (v[use] / a[use]).astype(np.float32)
    N = int(n.sum())
    vr = float(np.sqrt(np.sum(n[n > 0].astype(np.float64) * v[n > 0].astype(np.float64) ** 2) / N)) if N else 0.0
    am = float(a[n > 0].max()) if N else 0.0
    rg = vr / am if am > 0 else 0.0
    rmin = float(q.min()) if q.size else 0.0
    out = {"ratio_cell_min": rmin, "ratio_cell_max": float(q.max()) if q.size else 0.0, "ratio_global": rg,
           "ratio_criterion2": max(rg, rmin), "vrms_global": vr, "amax_global": am, "cells_used": int(use.sum()),
           "vmax": float(vmax) if vmax is not None else 0.0}
    out["drift_limit"] = 0.8 * (float(box) / K) / out["vmax"] if out["vmax"] > 0 else float("inf")
    return out


def interactions(cell_count, K: int, R: int, sink_plane_lo: int = 0, sink_plane_hi=None) -> int:
    """I = sum_c n_c sum_{c' in N(c)} n_c' (ordered pairs, self pairs included)."""
    lib = _load()
    cc = np.ascontiguousarray(cell_count, dtype=np.uint32)
    hi = int(K) if sink_plane_hi is None else int(sink_plane_hi)
    return int(lib.nfo_interactions(cc.ctypes.data_as(ctypes.POINTER(ctypes.c_uint32)), int(K), int(R),
                                    int(sink_plane_lo), hi))


def spline_over_r(r: float, eps: float) -> float:
    """|F|/r of Eq. 2."""
    return float(_load().nfo_spline_over_r(float(r), float(eps)))


def plummer_over_r(r: float, eps_p: float) -> float:
    """|F|/r of Eq. 1."""
    return float(_load().nfo_plummer_over_r(float(r), float(eps_p)))


def parity_error(a_test, a_ref):
    """Per-particle error metric of BASELINE.json's north_star:
    e_i = |a_test,i - a_ref,i| / max(|a_ref,i|, rms_k |a_ref,k|)   (2-norms over xyz).
    Modelled on the paper's own single-vs-double comparison."""
    a_test = np.asarray(a_test, dtype=np.float64)
    a_ref = np.asarray(a_ref, dtype=np.float64)
    mag = np.sqrt((a_ref ** 2).sum(axis=1))
    rms = np.sqrt((mag ** 2).mean()) if mag.size else 0.0
    den = np.maximum(mag, rms)
    den = np.where(den > 0, den, 1.0)
    return np.sqrt(((a_test - a_ref) ** 2).sum(axis=1)) / den
