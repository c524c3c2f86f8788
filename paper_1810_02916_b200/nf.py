"""Thin Python binding over the C-ABI library libnf.so (include/nf.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of csrc/.
PyTorch is used for device memory and streams.  There is NO CPU fallback: if libnf.so is
missing or no CUDA device is present, the constructor raises.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import List, Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnf.so")

NF_OK, NF_ERR_ARG, NF_ERR_NOMEM, NF_ERR_CUDA, NF_ERR_RANGE = 0, 1, 2, 3, 4
SOFT_SPLINE, SOFT_PLUMMER = 0, 1
NF_MASS_W = 0x100
NF_DENSE_ORDER = 0x200
_SOFT = {"spline": SOFT_SPLINE, "plummer": SOFT_PLUMMER}

def _soft_code(softening: str) -> int:
    """'spline' or 'plummer', optionally followed by '+dense' (NF_DENSE_ORDER: in-cell ordering of dense cells)."""
    base, _, opt = softening.partition("+")
    assert opt in ("", "dense"), softening
    return _SOFT[base] | (NF_DENSE_ORDER if opt else 0)


# every symbol include/nf.h declares
EXPORTS = ["nf_version", "nf_create", "nf_destroy", "nf_last_error", "nf_reserve", "nf_bin",
           "nf_out_of_range", "nf_forces", "nf_interactions", "nf_spline_equivalent_eps",
           "nf_stream_slabs", "nf_last_forces_timing", "nf_launch_count", "nf_forces_host", "nf_reserve_host",
           "nf_bin_m", "nf_forces_ex", "nf_kick_drift", "nf_cell_vrms", "nf_stream_step_slabs",
           "nf_keys", "nf_forces_chunk", "nf_forces_host_m", "nf_regroup_plane", "nf_stream_step_regroup",
           "nf_forces_host_begin", "nf_forces_host_end", "nf_timestep_terms", "nf_forces_tree", "nf_tree_stats", "nf_last_tree_timing",
           "nf_timestep_terms_static"]


class NFError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libnf status {status}: {msg}")
        self.status = status


class TimeStep(ctypes.Structure):
    _fields_ = [("ratio_cell_min", ctypes.c_double), ("ratio_cell_max", ctypes.c_double), ("ratio_global", ctypes.c_double),
                ("ratio_criterion2", ctypes.c_double), ("vrms_global", ctypes.c_double), ("amax_global", ctypes.c_double),
                ("vmax", ctypes.c_double), ("drift_limit", ctypes.c_double), ("cells_used", ctypes.c_int64)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class StreamStats(ctypes.Structure):
    _fields_ = [("particles_in", ctypes.c_int64), ("particles_out", ctypes.c_int64),
                ("interactions", ctypes.c_int64), ("out_of_range", ctypes.c_int64),
                ("h2d_bytes", ctypes.c_double), ("d2h_bytes", ctypes.c_double),
                ("h2d_seconds", ctypes.c_double), ("d2h_seconds", ctypes.c_double),
                ("kernel_seconds", ctypes.c_double), ("wall_seconds", ctypes.c_double),
                ("h2d_gbps", ctypes.c_double), ("d2h_gbps", ctypes.c_double),
                ("overlap_fraction", ctypes.c_double), ("force_seconds", ctypes.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def load_library(path: str = LIB_PATH) -> ctypes.CDLL:
    """dlopen libnf.so and declare the prototypes of include/nf.h.  Raises if it is missing:
    build it with ``python -m paper_1810_02916_b200.build``."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not found: run `python -m paper_1810_02916_b200.build` (no CPU fallback exists)")
    lib = ctypes.CDLL(path)
    vp, i32, i64, f32 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_float
    lib.nf_version.restype = i32
    lib.nf_create.restype = i32
    lib.nf_create.argtypes = [ctypes.POINTER(vp), i32]
    lib.nf_destroy.restype = i32
    lib.nf_destroy.argtypes = [vp]
    lib.nf_last_error.restype = ctypes.c_char_p
    lib.nf_last_error.argtypes = [vp]
    lib.nf_reserve.restype = i32
    lib.nf_reserve.argtypes = [vp, i64, i32]
    lib.nf_bin.restype = i32
    lib.nf_bin.argtypes = [vp, vp, i64, i32, f32, vp, vp, vp, vp, vp]
    lib.nf_bin_m.restype = i32
    lib.nf_bin_m.argtypes = [vp, vp, vp, i64, i32, f32, vp, vp, vp, vp, vp]
    lib.nf_forces_ex.restype = i32
    lib.nf_forces_ex.argtypes = [vp, vp, vp, vp, vp, i64, i32, i32, f32, f32, f32, i32, vp, vp, vp]
    lib.nf_forces_tree.restype = i32
    lib.nf_forces_tree.argtypes = [vp, vp, vp, vp, i64, i32, i32, f32, f32, f32, i32, f32, vp, vp, vp]
    lib.nf_last_tree_timing.restype = i32
    lib.nf_last_tree_timing.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    lib.nf_tree_stats.restype = i32
    lib.nf_tree_stats.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i64), vp]
    lib.nf_kick_drift.restype = i32
    lib.nf_kick_drift.argtypes = [vp, vp, vp, vp, i64, f32, f32, f32, vp]
    lib.nf_cell_vrms.restype = i32
    lib.nf_cell_vrms.argtypes = [vp, vp, vp, vp, i64, i32, vp, vp, vp]
    lib.nf_timestep_terms.restype = i32
    lib.nf_timestep_terms.argtypes = [vp, vp, vp, vp, i32, f32, vp, ctypes.POINTER(TimeStep), vp]
    lib.nf_timestep_terms_static.restype = i32
    lib.nf_timestep_terms_static.argtypes = [vp, vp, vp, vp, i32, f32, vp, ctypes.POINTER(TimeStep), vp]
    lib.nf_out_of_range.restype = i32
    lib.nf_out_of_range.argtypes = [vp, ctypes.POINTER(i64), vp]
    lib.nf_forces.restype = i32
    lib.nf_forces.argtypes = [vp, vp, vp, vp, vp, i64, i32, i32, f32, f32, f32, i32, vp, vp]
    lib.nf_interactions.restype = i32
    lib.nf_interactions.argtypes = [vp, vp, i32, i32, ctypes.POINTER(i64), vp]
    lib.nf_spline_equivalent_eps.restype = f32
    lib.nf_spline_equivalent_eps.argtypes = [f32]
    lib.nf_stream_slabs.restype = i32
    lib.nf_stream_slabs.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(i64), i32, i32, i32, f32, f32, i32, f32,
                                    i32, ctypes.POINTER(vp), ctypes.POINTER(StreamStats), vp]
    lib.nf_stream_step_slabs.restype = i32
    lib.nf_stream_step_slabs.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(i64), i32, i32, i32, f32, f32,
                                         i32, f32, i32, f32, f32, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(vp),
                                         ctypes.POINTER(StreamStats), vp]
    lib.nf_last_forces_timing.restype = i32
    lib.nf_last_forces_timing.argtypes = [vp, ctypes.POINTER(f32), ctypes.POINTER(f32)]
    lib.nf_forces_host.restype = i32
    lib.nf_forces_host.argtypes = [vp, vp, i64, i32, i32, f32, f32, f32, i32, vp, vp]
    lib.nf_reserve_host.restype = i32
    lib.nf_reserve_host.argtypes = [vp, i64, i32]
    lib.nf_forces_host_m.restype = i32
    lib.nf_forces_host_m.argtypes = [vp, vp, vp, i64, i32, i32, f32, f32, f32, i32, vp, vp]
    lib.nf_regroup_plane.restype = i32
    lib.nf_regroup_plane.argtypes = [vp, vp, vp, i64, i32, f32, i32, vp, vp, ctypes.POINTER(i64), vp]
    lib.nf_stream_step_regroup.restype = i32
    lib.nf_stream_step_regroup.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(i64), i32, i32, i32, f32, f32,
                                           i32, f32, i32, f32, f32, ctypes.POINTER(vp), ctypes.POINTER(vp), ctypes.POINTER(i64),
                                           ctypes.POINTER(vp), ctypes.POINTER(StreamStats), vp]
    lib.nf_forces_host_begin.restype = i32
    lib.nf_forces_host_begin.argtypes = [vp, vp, i64, i32, i32, f32, f32, f32, i32, vp, vp]
    lib.nf_forces_host_end.restype = i32
    lib.nf_forces_host_end.argtypes = [vp]
    lib.nf_keys.restype = i32
    lib.nf_keys.argtypes = [vp, vp, i64, i32, f32, vp, vp]
    lib.nf_forces_chunk.restype = i32
    lib.nf_forces_chunk.argtypes = [vp, vp, vp, vp, i64, i32, i32, f32, f32, f32, i32, i32, i32, vp, vp, vp]
    lib.nf_launch_count.restype = i32
    lib.nf_launch_count.argtypes = [vp, ctypes.POINTER(i64)]
    _lib = lib
    return lib


@dataclass
class Binned:
    """Output of nf_bin (all device tensors)."""
    pos_sorted: torch.Tensor   # float32 [N, 4]: cell-centred offsets, w = 0
    perm: torch.Tensor         # int32 view of uint32 [N]
    cell_count: torch.Tensor   # int32 view of uint32 [K^3]
    cell_offset: torch.Tensor  # int64 view of uint64 [K^3 + 1]
    N: int
    K: int
    box: float


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    return None if t is None else t.data_ptr()


class Context:
    """nf_create / nf_destroy."""

    def __init__(self, device: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1810_02916_b200.nf needs a CUDA device (there is no CPU fallback)")
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        self._h = ctypes.c_void_p()
        torch.cuda.init()
        with torch.cuda.device(self.device):
            torch.zeros(1, device=self.device)      # make sure the primary context exists
            rc = self.lib.nf_create(ctypes.byref(self._h), device)
        if rc != NF_OK:
            raise NFError(rc, "nf_create failed")

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self.lib.nf_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, allow=()):
        if rc != NF_OK and rc not in allow:
            raise NFError(rc, self.lib.nf_last_error(self._h).decode())
        return rc

    def _stream(self, stream: Optional[torch.cuda.Stream]):
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        return ctypes.c_void_p(s.cuda_stream)

    def reserve(self, maxN: int, K: int):
        self._check(self.lib.nf_reserve(self._h, int(maxN), int(K)))

    def bin(self, pos: torch.Tensor, K: int, box: float, out: Optional[Binned] = None, stream=None,
            mass: Optional[torch.Tensor] = None) -> Binned:
        """nf_bin (nf_bin_m when ``mass`` float32 [N] is given: it lands in pos_sorted[:, 3]): pos float32
        [N, 3] on the device -> cell-contiguous arrays (written into ``out`` if given, so repeated
        calls reuse the same device buffers)."""
        assert pos.is_cuda and pos.dtype == torch.float32 and pos.dim() == 2 and pos.shape[1] == 3 and pos.is_contiguous()
        N = pos.shape[0]
        dev = pos.device
        ncell = int(K) ** 3
        if out is None:
            out = Binned(torch.empty(N, 4, dtype=torch.float32, device=dev),
                         torch.empty(N, dtype=torch.int32, device=dev),
                         torch.empty(ncell, dtype=torch.int32, device=dev),
                         torch.empty(ncell + 1, dtype=torch.int64, device=dev), N, int(K), float(box))
        assert out.N == N and out.K == int(K) and out.box == float(box)
        if mass is not None:
            assert mass.is_cuda and mass.dtype == torch.float32 and mass.shape == (N,) and mass.is_contiguous()
            self._check(self.lib.nf_bin_m(self._h, _ptr(pos), _ptr(mass), N, int(K), float(box), _ptr(out.pos_sorted),
                                          _ptr(out.perm), _ptr(out.cell_count), _ptr(out.cell_offset), self._stream(stream)))
            return out
        self._check(self.lib.nf_bin(self._h, _ptr(pos), N, int(K), float(box), _ptr(out.pos_sorted), _ptr(out.perm),
                                    _ptr(out.cell_count), _ptr(out.cell_offset), self._stream(stream)))
        return out

    def out_of_range(self, stream=None) -> int:
        n = ctypes.c_int64(0)
        self._check(self.lib.nf_out_of_range(self._h, ctypes.byref(n), self._stream(stream)), allow=(NF_ERR_RANGE,))
        return int(n.value)

    def keys(self, pos: torch.Tensor, K: int, box: float, stream=None) -> torch.Tensor:
        """nf_keys: cell key (cx*K+cy)*K+cz per particle as an int32 view of uint32 [N]; the x-plane is key // K^2."""
        assert pos.is_cuda and pos.dtype == torch.float32 and pos.dim() == 2 and pos.shape[1] == 3 and pos.is_contiguous()
        out = torch.empty(pos.shape[0], dtype=torch.int32, device=pos.device)
        self._check(self.lib.nf_keys(self._h, _ptr(pos), pos.shape[0], int(K), float(box), _ptr(out), self._stream(stream)))
        return out

    def forces_chunk(self, b: Binned, R: int, eps: float, Gm: float, x_lo: int, x_hi: int, softening: str = "spline",
                     original_order: bool = True, out: Optional[torch.Tensor] = None, stream=None,
                     use_mass: bool = False, cell_amax: Optional[torch.Tensor] = None, dense_order: bool = False) -> torch.Tensor:
        """nf_forces_chunk: accelerations of the particles in x-planes [x_lo, x_hi) only (rows of the other
        particles -- ghosts -- are left untouched); every particle of ``b`` acts as a source."""
        acc = out if out is not None else torch.zeros(b.N, 3, dtype=torch.float32, device=b.pos_sorted.device)
        assert acc.is_cuda and acc.dtype == torch.float32 and acc.shape == (b.N, 3) and acc.is_contiguous()
        self._check(self.lib.nf_forces_chunk(self._h, _ptr(b.pos_sorted), _ptr(b.cell_offset),
                                             _ptr(b.perm) if original_order else None, b.N, b.K, int(R), float(eps),
                                             float(b.box), float(Gm),
                                             _soft_code(softening) | (NF_MASS_W if use_mass else 0) | (NF_DENSE_ORDER if dense_order else 0),
                                             int(x_lo), int(x_hi), _ptr(acc), _ptr(cell_amax), self._stream(stream)))
        return acc

    def forces(self, b: Binned, R: int, eps: float, Gm: float, softening: str = "spline",
               original_order: bool = True, out: Optional[torch.Tensor] = None, stream=None,
               use_mass: bool = False, cell_amax: Optional[torch.Tensor] = None, dense_order: bool = False) -> torch.Tensor:
        """nf_forces: accelerations float32 [N, 3] (caller's order if original_order).
        use_mass: sources carry their masses in pos_sorted[:, 3] (NF_MASS_W; Gm is then G).
        dense_order: NF_DENSE_ORDER, the in-cell ordering of dense cells (automatic when N / K^3 >= 512).
        cell_amax: float32 [K^3] device tensor to receive the per-cell max |a| (nf_forces_ex)."""
        acc = out if out is not None else torch.empty(b.N, 3, dtype=torch.float32, device=b.pos_sorted.device)
        assert acc.is_cuda and acc.dtype == torch.float32 and acc.shape == (b.N, 3) and acc.is_contiguous()
        if use_mass or cell_amax is not None or dense_order:
            if cell_amax is not None:
                assert cell_amax.is_cuda and cell_amax.dtype == torch.float32 and cell_amax.numel() == b.K ** 3 and cell_amax.is_contiguous()
            self._check(self.lib.nf_forces_ex(self._h, _ptr(b.pos_sorted), _ptr(b.cell_offset), _ptr(b.cell_count),
                                              _ptr(b.perm) if original_order else None, b.N, b.K, int(R), float(eps),
                                              float(b.box), float(Gm),
                                              _soft_code(softening) | (NF_MASS_W if use_mass else 0) | (NF_DENSE_ORDER if dense_order else 0),
                                              _ptr(acc), _ptr(cell_amax), self._stream(stream)))
            return acc
        self._check(self.lib.nf_forces(self._h, _ptr(b.pos_sorted), _ptr(b.cell_offset), _ptr(b.cell_count),
                                       _ptr(b.perm) if original_order else None, b.N, b.K, int(R), float(eps),
                                       float(b.box), float(Gm), _soft_code(softening), _ptr(acc), self._stream(stream)))
        return acc

    def forces_tree(self, b: Binned, R: int, eps: float, Gm: float, theta: float, softening: str = "spline",
                    original_order: bool = True, out: Optional[torch.Tensor] = None, stream=None, use_mass: bool = False,
                    cell_amax: Optional[torch.Tensor] = None) -> torch.Tensor:
        """nf_forces_tree: nf_forces_ex with the sources of dense cells (>= 4096 particles) met through a tree with
        opening angle theta (readings t1-t6).  theta = 0 is the direct sum."""
        acc = out if out is not None else torch.empty(b.N, 3, dtype=torch.float32, device=b.pos_sorted.device)
        assert acc.is_cuda and acc.dtype == torch.float32 and acc.shape == (b.N, 3) and acc.is_contiguous()
        if cell_amax is not None:
            assert cell_amax.is_cuda and cell_amax.dtype == torch.float32 and cell_amax.numel() == b.K ** 3 and cell_amax.is_contiguous()
        self._check(self.lib.nf_forces_tree(self._h, _ptr(b.pos_sorted), _ptr(b.cell_offset), _ptr(b.perm) if original_order else None,
                                            b.N, b.K, int(R), float(eps), float(b.box), float(Gm),
                                            _soft_code(softening) | (NF_MASS_W if use_mass else 0), float(theta),
                                            _ptr(acc), _ptr(cell_amax), self._stream(stream)))
        return acc

    def last_tree_timing(self) -> float:
        """Milliseconds of the walk kernel of the last forces_tree (CUDA events on its stream)."""
        t = ctypes.c_float(0)
        self._check(self.lib.nf_last_tree_timing(self._h, ctypes.byref(t)))
        return float(t.value)

    def tree_stats(self, stream=None) -> dict:
        """nf_tree_stats: (sink, accepted node) and (sink, particle of an opened leaf) pairs of the last forces_tree."""
        a, b_ = ctypes.c_int64(0), ctypes.c_int64(0)
        self._check(self.lib.nf_tree_stats(self._h, ctypes.byref(a), ctypes.byref(b_), self._stream(stream)))
        return {"node": int(a.value), "leaf": int(b_.value)}

    def kick_drift(self, pos: torch.Tensor, vel: torch.Tensor, acc: torch.Tensor, kick: float, drift: float,
                   box: float, stream=None):
        """nf_kick_drift: v += a*kick; x = wrap(x + v*drift), in place on float32 [N, 3] device tensors."""
        for t in (pos, vel, acc):
            assert t.is_cuda and t.dtype == torch.float32 and t.dim() == 2 and t.shape[1] == 3 and t.is_contiguous()
        assert pos.shape == vel.shape == acc.shape
        self._check(self.lib.nf_kick_drift(self._h, _ptr(pos), _ptr(vel), _ptr(acc), pos.shape[0], float(kick),
                                           float(drift), float(box), self._stream(stream)))

    def cell_vrms(self, vel: torch.Tensor, b: Binned, original_order: bool = True, stream=None):
        """nf_cell_vrms: (per-cell rms speed float32 [K^3], max |v_axis| float32 [1]) for velocities in the
        caller's order (or in nf_bin's sorted order if not original_order)."""
        assert vel.is_cuda and vel.dtype == torch.float32 and vel.shape == (b.N, 3) and vel.is_contiguous()
        vrms = torch.empty(b.K ** 3, dtype=torch.float32, device=vel.device)
        vmax = torch.empty(1, dtype=torch.float32, device=vel.device)
        self._check(self.lib.nf_cell_vrms(self._h, _ptr(vel), _ptr(b.perm) if original_order else None, _ptr(b.cell_offset),
                                          b.N, b.K, _ptr(vrms), _ptr(vmax), self._stream(stream)))
        return vrms, vmax

    def timestep_terms(self, cell_vrms: torch.Tensor, cell_amax: torch.Tensor, b: Binned, vmax: Optional[torch.Tensor] = None,
                       stream=None) -> dict:
        """nf_timestep_terms: the reduction of time-step criteria 2 and 3 over the cells."""
        ncell = b.K ** 3
        for t in (cell_vrms, cell_amax):
            assert t.is_cuda and t.dtype == torch.float32 and t.numel() == ncell and t.is_contiguous()
        ts = TimeStep()
        self._check(self.lib.nf_timestep_terms(self._h, _ptr(cell_vrms), _ptr(cell_amax), _ptr(b.cell_offset), b.K, float(b.box),
                                               _ptr(vmax) if vmax is not None else None, ctypes.byref(ts), self._stream(stream)))
        return ts.as_dict()

    def timestep_terms_static(self, cell_vrms: torch.Tensor, cell_amax: torch.Tensor, b: Binned, vmax: Optional[torch.Tensor] = None,
                              stream=None) -> dict:
        """nf_timestep_terms_static: timestep_terms with its scratch in a fixed __device__ array -- no allocation; K <= 256;
        calls that overlap on the GPU race (include/nf.h)."""
        ncell = b.K ** 3
        for t in (cell_vrms, cell_amax):
            assert t.is_cuda and t.dtype == torch.float32 and t.numel() == ncell and t.is_contiguous()
        ts = TimeStep()
        self._check(self.lib.nf_timestep_terms_static(self._h, _ptr(cell_vrms), _ptr(cell_amax), _ptr(b.cell_offset), b.K, float(b.box),
                                               _ptr(vmax) if vmax is not None else None, ctypes.byref(ts), self._stream(stream)))
        return ts.as_dict()

    def reserve_host(self, maxN: int, K: int):
        self._check(self.lib.nf_reserve_host(self._h, int(maxN), int(K)))

    def forces_host(self, pos_host: torch.Tensor, K: int, R: int, eps: float, box: float, Gm: float,
                    softening: str = "spline", out: Optional[torch.Tensor] = None, stream=None,
                    mass_host: Optional[torch.Tensor] = None, strict: bool = False) -> torch.Tensor:
        """nf_forces_host (nf_forces_host_m when ``mass_host`` float32 [N] is given): the whole path from a
        HOST float32 [N, 3] tensor (pinned recommended) to a host float32 [N, 3] acceleration tensor; H2D,
        binning, forces and D2H all inside the call.  strict: raise on NF_ERR_RANGE instead of returning."""
        assert (not pos_host.is_cuda) and pos_host.dtype == torch.float32 and pos_host.dim() == 2 \
            and pos_host.shape[1] == 3 and pos_host.is_contiguous()
        N = pos_host.shape[0]
        if out is None:
            out = torch.empty(N, 3, dtype=torch.float32).pin_memory()
        assert (not out.is_cuda) and out.dtype == torch.float32 and out.shape == (N, 3) and out.is_contiguous()
        allow = () if strict else (NF_ERR_RANGE,)
        if mass_host is not None:
            assert (not mass_host.is_cuda) and mass_host.dtype == torch.float32 and mass_host.shape == (N,) and mass_host.is_contiguous()
            self._check(self.lib.nf_forces_host_m(self._h, _ptr(pos_host), _ptr(mass_host), N, int(K), int(R), float(eps),
                                                  float(box), float(Gm), _soft_code(softening) | NF_MASS_W, _ptr(out),
                                                  self._stream(stream)), allow=allow)
            return out
        self._check(self.lib.nf_forces_host(self._h, _ptr(pos_host), N, int(K), int(R), float(eps), float(box),
                                            float(Gm), _soft_code(softening), _ptr(out), self._stream(stream)), allow=allow)
        return out

    def forces_host_begin(self, pos_host: torch.Tensor, K: int, R: int, eps: float, box: float, Gm: float, out: torch.Tensor,
                          softening: str = "spline", stream=None):
        """nf_forces_host_begin: enqueue one whole step from pinned host positions into the pinned host tensor
        ``out``; returns at once (at most two steps in flight).  Pair with forces_host_end()."""
        for t in (pos_host, out):
            assert (not t.is_cuda) and t.dtype == torch.float32 and t.dim() == 2 and t.shape[1] == 3 and t.is_contiguous() and t.is_pinned()
        assert out.shape == pos_host.shape
        self._check(self.lib.nf_forces_host_begin(self._h, _ptr(pos_host), pos_host.shape[0], int(K), int(R), float(eps), float(box),
                                                  float(Gm), _soft_code(softening), _ptr(out), self._stream(stream)))

    def forces_host_end(self, strict: bool = False):
        """nf_forces_host_end: wait for the oldest step in flight; its ``out`` tensor is then complete."""
        return self._check(self.lib.nf_forces_host_end(self._h), allow=() if strict else (NF_ERR_RANGE,))

    def interactions(self, b: Binned, R: int, stream=None) -> int:
        n = ctypes.c_int64(0)
        self._check(self.lib.nf_interactions(self._h, _ptr(b.cell_count), b.K, int(R), ctypes.byref(n), self._stream(stream)))
        return int(n.value)

    def last_forces_timing(self):
        """(kernel_ms, total_ms) of the last forces() call, from CUDA events on its stream."""
        k, t = ctypes.c_float(0), ctypes.c_float(0)
        self._check(self.lib.nf_last_forces_timing(self._h, ctypes.byref(k), ctypes.byref(t)))
        return float(k.value), float(t.value)

    def launch_count(self) -> int:
        """Kernels launched by this context so far (host counter)."""
        n = ctypes.c_int64(0)
        self._check(self.lib.nf_launch_count(self._h, ctypes.byref(n)))
        return int(n.value)

    def stream_slabs(self, planes: Sequence[torch.Tensor], P: int, K: int, R: int, eps: float, box: float,
                     plane0: int, Gm: float, softening: str = "spline",
                     out: Optional[List[torch.Tensor]] = None, stream=None, strict: bool = True):
        """nf_stream_slabs: planes = P + 2R pinned host float32 [n_q, 3] tensors; returns
        (list of P pinned host float32 [n, 3] acceleration tensors, stats dict).  NF_ERR_RANGE
        (mis-filed or out-of-range particles, counted in stats["out_of_range"]) raises unless
        strict is False."""
        NP = P + 2 * R
        assert len(planes) == NP
        for t in planes:
            assert (not t.is_cuda) and t.dtype == torch.float32 and t.dim() == 2 and t.shape[1] == 3 and t.is_contiguous()
            assert t.shape[0] == 0 or t.is_pinned(), "plane tensors must be pinned host memory"
        if out is None:
            out = [torch.empty(planes[R + p].shape[0], 3, dtype=torch.float32).pin_memory() for p in range(P)]
        pos_ptrs = (ctypes.c_void_p * NP)(*[t.data_ptr() if t.shape[0] else None for t in planes])
        ns = (ctypes.c_int64 * NP)(*[t.shape[0] for t in planes])
        acc_ptrs = (ctypes.c_void_p * P)(*[t.data_ptr() if t.shape[0] else None for t in out])
        stats = StreamStats()
        self._check(self.lib.nf_stream_slabs(self._h, pos_ptrs, ns, int(P), int(K), int(R), float(eps), float(box),
                                             int(plane0), float(Gm), _soft_code(softening), acc_ptrs, ctypes.byref(stats),
                                             self._stream(stream)), allow=() if strict else (NF_ERR_RANGE,))
        return out, stats.as_dict()

    def stream_step_slabs(self, planes, vels, P, K, R, eps, box, plane0, Gm, kick, drift, softening="spline", want_acc=False, stream=None):
        """nf_stream_step_slabs: planes = P + 2R pinned float32 [n_q, 3] position tensors, vels = P pinned
        velocity tensors of the sink planes; returns (new positions, new velocities, accelerations or None,
        stats), each a list of P pinned host tensors."""
        NP = P + 2 * R
        assert len(planes) == NP and len(vels) == P
        for t in list(planes) + list(vels):
            assert (not t.is_cuda) and t.dtype == torch.float32 and t.dim() == 2 and t.shape[1] == 3 and t.is_contiguous()
            assert t.shape[0] == 0 or t.is_pinned(), "plane tensors must be pinned host memory"
        mk = lambda: [torch.empty(planes[R + p].shape[0], 3, dtype=torch.float32).pin_memory() for p in range(P)]
        pos_out, vel_out, acc = mk(), mk(), (mk() if want_acc else None)
        tab = lambda ts: (ctypes.c_void_p * len(ts))(*[t.data_ptr() if t.shape[0] else None for t in ts])
        ns = (ctypes.c_int64 * NP)(*[t.shape[0] for t in planes])
        stats = StreamStats()
        self._check(self.lib.nf_stream_step_slabs(self._h, tab(planes), tab(vels), ns, int(P), int(K), int(R), float(eps), float(box),
                                                  int(plane0), float(Gm), _soft_code(softening), float(kick), float(drift),
                                                  tab(pos_out), tab(vel_out), tab(acc) if acc is not None else None,
                                                  ctypes.byref(stats), self._stream(stream)))
        return pos_out, vel_out, acc, stats.as_dict()


    def regroup_plane(self, pos: torch.Tensor, vel: torch.Tensor, K: int, box: float, plane_cx: int, stream=None, strict: bool = True):
        """nf_regroup_plane: (positions, velocities) of one drifted plane as [to plane-1 | stay | to plane+1]
        and the three segment lengths."""
        for t in (pos, vel):
            assert t.is_cuda and t.dtype == torch.float32 and t.dim() == 2 and t.shape[1] == 3 and t.is_contiguous()
        assert pos.shape == vel.shape
        po, vo = torch.empty_like(pos), torch.empty_like(vel)
        seg = (ctypes.c_int64 * 3)()
        self._check(self.lib.nf_regroup_plane(self._h, _ptr(pos), _ptr(vel), pos.shape[0], int(K), float(box), int(plane_cx),
                                              _ptr(po), _ptr(vo), seg, self._stream(stream)), allow=() if strict else (NF_ERR_RANGE,))
        return po, vo, [int(x) for x in seg]

    def stream_step_regroup(self, seg_pos, seg_vel, P, K, R, eps, box, plane0, Gm, kick, drift, softening="spline",
                            out_pos=None, out_vel=None, want_acc=False, stream=None, strict: bool = True):
        """nf_stream_step_regroup.  seg_pos: P + 2R planes, each a list of up to 3 pinned float32 [n, 3]
        segments (None or empty = nothing); seg_vel: the same for the P sink planes.  Returns (out_pos, out_vel:
        P pinned tensors holding each sink plane's drifted particles as [to plane-1 | stay | to plane+1],
        seg_n: P lists of 3 lengths, accelerations or None, stats)."""
        NP = P + 2 * R
        assert len(seg_pos) == NP and len(seg_vel) == P

        def table(planes):
            ptrs, ns = [], []
            for segs in planes:
                segs = list(segs) + [None] * (3 - len(segs))
                assert len(segs) == 3
                for t in segs:
                    if t is None or t.shape[0] == 0:
                        ptrs.append(None); ns.append(0)
                        continue
                    assert (not t.is_cuda) and t.dtype == torch.float32 and t.dim() == 2 and t.shape[1] == 3 and t.is_contiguous()
                    assert t.is_pinned(), "plane segments must be pinned host memory"
                    ptrs.append(t.data_ptr()); ns.append(t.shape[0])
            return (ctypes.c_void_p * len(ptrs))(*ptrs), ns
        pos_ptrs, pos_ns = table(seg_pos)
        vel_ptrs, vel_ns = table(seg_vel)
        assert vel_ns == pos_ns[3 * R:3 * (R + P)], "velocity segments must match the sink planes' position segments"
        n_sink = [sum(pos_ns[3 * (R + p):3 * (R + p) + 3]) for p in range(P)]
        mk = lambda: [torch.empty(n, 3, dtype=torch.float32).pin_memory() for n in n_sink]
        out_pos = out_pos if out_pos is not None else mk()
        out_vel = out_vel if out_vel is not None else mk()
        acc = mk() if want_acc else None
        for p in range(P):
            assert out_pos[p].shape[0] >= n_sink[p] and out_vel[p].shape[0] >= n_sink[p]
        tab = lambda ts: (ctypes.c_void_p * len(ts))(*[t.data_ptr() if t.shape[0] else None for t in ts])
        ns = (ctypes.c_int64 * len(pos_ns))(*pos_ns)
        out_n = (ctypes.c_int64 * (3 * P))()
        stats = StreamStats()
        self._check(self.lib.nf_stream_step_regroup(self._h, pos_ptrs, vel_ptrs, ns, int(P), int(K), int(R), float(eps), float(box),
                                                    int(plane0), float(Gm), _soft_code(softening), float(kick), float(drift),
                                                    tab(out_pos), tab(out_vel), out_n, tab(acc) if acc is not None else None,
                                                    ctypes.byref(stats), self._stream(stream)),
                    allow=() if strict else (NF_ERR_RANGE,))
        seg_n = [[int(out_n[3 * p + k]) for k in range(3)] for p in range(P)]
        return out_pos, out_vel, seg_n, acc, stats.as_dict()


def spline_equivalent_eps(eps_plummer: float) -> float:
    return float(load_library().nf_spline_equivalent_eps(float(eps_plummer)))
