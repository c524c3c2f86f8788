"""Helpers shared by the GPU parity tests (test infrastructure; may call the oracle)."""
import numpy as np
import torch

import oracle


def oracle_plane_of(K: int, box: float):
    """``plane_of`` for inputs.make_slab_planes: the x-plane each particle is filed under, taken from
    the ORACLE's cell assignment (keys // K^2), so that no test input depends on the CUDA path."""
    def plane_of(x: torch.Tensor) -> torch.Tensor:
        keys, _ = oracle.keys(x.detach().cpu().numpy(), K, box)
        return torch.from_numpy((keys // np.uint32(K * K)).astype(np.int64)).to(x.device)
    return plane_of


def frac_error(a_test, a_ref):
    """The paper's own statistic: fractional error |da| / |a| per particle."""
    a_test = np.asarray(a_test, dtype=np.float64)
    a_ref = np.asarray(a_ref, dtype=np.float64)
    mag = np.sqrt((a_ref ** 2).sum(axis=1))
    return np.sqrt(((a_test - a_ref) ** 2).sum(axis=1)) / np.where(mag > 0, mag, 1.0)
