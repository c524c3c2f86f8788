"""B200-native near-field force of the Abacus N-body method (arXiv:1810.02916, Sec. 2.1).

Public API (thin argument marshalling over the C-ABI library ``libnf.so`` declared in
``include/nf.h``; every step of the path runs in hand-written CUDA kernels for sm_100a):

    from paper_1810_02916_b200 import nf
    ctx = nf.Context()                      # nf_create
    b = ctx.bin(pos, K, box)                # nf_bin      (device tensors in/out)
    acc = ctx.forces(b, R, eps, Gm)         # nf_forces
    ctx.stream_slabs(...)                   # nf_stream_slabs (pinned host in/out)

Importing this package does not load the CUDA library; ``nf`` loads it on first use and
raises if it is missing (there is no CPU fallback).  ``inputs`` holds the seeded synthetic
input generators shared by the tests, the benchmark and the oracle's callers; it contains
none of the method's arithmetic.
"""
__all__ = ["nf", "inputs"]
__version__ = "0.1.0"
